// dslash.cu -- the even/odd staggered Dirac operator D_eo / D_oe (Eq. 7;
// the paper's acc_Deo of Listing 2), hand-written for sm_100a.
//
//   (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+ U_mu(x) psi(x+mu) - s- U_mu(x-mu)^dagger psi(x-mu) ]
//
// Steps a2-a5 of SURVEY.md section 8(a); readings R1-R5, R8, R9 of DESIGN.md.
//   a2  one thread per output site; coordinates, the 8 neighbour half-indices, eta_mu(x) and the
//       antiperiodic sign come from integer arithmetic on the thread index (no neighbour tables,
//       unlike the paper's nnp_openacc/nnm_openacc)
//   a3  each link is read exactly once per application with streaming (evict-first) loads; with
//       2-row storage the third row is rebuilt in registers, r2 = (r0 ^ r1)^*
//   a4  8 SU(3) x colour-vector products accumulated in registers, one store per site
//   a5  optional fused epilogue out = coef*x - D in (Eq. 8) and the partial sums of
//       Re<x,out> for CG, reduced deterministically (reduce.cuh)
// The kernel is bound by HBM bandwidth (1248 B/site fp64 18-real vs 570 flop/site): no tensor cores.
#include "reduce.cuh"

#include "peer.cuh"
#include "su3.cuh"

// MODE 0: out = D in;  1: out = coef*x - D in;  2: as 1, plus Re<x,out> -> solver_after_pq
// BF != 0: every link enters as e^{i theta_mu(x)} U_mu(x) (the `backfield` argument of the paper's acc_Deo, Listing 2,
// PAPER.md:320-326; reading R6), [parity][mu][idxh]; the phase multiplies the neighbour vector together with
// eta / the boundary sign, AFTER the third row was rebuilt from the SU(3) link.  BF 1: theta stored, one real per
// link, sincos in-kernel; BF 2: (cos theta, sin theta) stored (option backfield_format).
// HALO 1 (slab mode over the peer transport, peer.cuh): [i_begin, i_end) are the owned slices; the kernel first
// waits for the two faces of `in` pushed by the neighbours and takes the x3 hops that leave the slab from the
// landing buffers instead of the vector's ghost slices; MODE 2 publishes the local <x,out> to every rank.
template <typename T, int LAYOUT, int RECON12, int MODE, int MINB, int POLICY, int BF, int HALO>
__global__ void __launch_bounds__(256, MINB)
dslash_kernel(const Geom g, const int parity, T *__restrict__ out, const T *__restrict__ in,
              const T *__restrict__ links, const T *__restrict__ xin, const double coef,
              SolverState *__restrict__ st, double *__restrict__ partials, const int gate,
              const int i_begin, const int i_end, const T *__restrict__ bf, const PeerDev *__restrict__ pdp,
              const int push_out)
{
    pdl_wait();
    pdl_trigger();
    if (gate) {
        int d = *(volatile int *)&st->done;
        if (d) {   // a converged solve: the rest of the enqueued iterations are no-ops
            if (gate == 2 && d == 1 && blockIdx.x == 0 && threadIdx.x == 0) st->done = 2;
            return;
        }
    }
    bool waited = false;
    int rot = 0;
    if (HALO) {
        // the push of `in` is the previous kernel of the stream: its stores have landed, tell the neighbours
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            peer_signal_halo(*pdp, 1 - parity);
            if (push_out) peer_bump_halo(*pdp, parity);      // this kernel pushes the faces of `out` itself (below)
        }
        // tiles start one slice in, so that the two boundary slices (the only tiles that wait) come last
        if (g.s3 % (int)blockDim.x == 0 && (int)(gridDim.x * blockDim.x) >= i_end - i_begin) rot = g.s3 / (int)blockDim.x;
    }
    double dot = 0.0;
    L2Pol pol = {0, 0};
    if (POLICY) pol = make_l2pol();
    const size_t Vh = (size_t)g.Vh;
    // One tile = blockDim.x consecutive sites.  gridDim.x = number of tiles (one pass), or fewer
    // CTAs that loop (option dslash_persist): the reduction protocol below is then paid once per
    // CTA instead of once per tile.
    // Sites [i_begin, i_end): the whole parity, or a range of x3 slices (lqcd_dslash_slices; slab mode).
    int bx = blockIdx.x + rot;
    if (bx >= (int)gridDim.x) bx -= gridDim.x;
    for (int tile0 = i_begin + bx * blockDim.x; tile0 < i_end; tile0 += gridDim.x * blockDim.x) {
    if (HALO && !waited && (tile0 < i_begin + g.s3 || tile0 + (int)blockDim.x > i_end - g.s3)) {
        // only tiles that touch a boundary slice read the faces: the interior computes while they arrive
        peer_wait_halo(*pdp, 1 - parity);
        waited = true;
    }
    const int i = tile0 + threadIdx.x;
    const bool valid = i < i_end;
    if (valid) {
        // ---- a2: site decode (Eq. 9), neighbours, phases ---------------------------------
        uint32_t t = fd_div((uint32_t)i, g.dNh0);
        const int hx0 = i - (int)t * g.Nh0;
        uint32_t t2 = fd_div(t, g.dN1);
        const int x1 = (int)t - (int)t2 * g.N1;
        const int x3 = (int)fd_div(t2, g.dN2);
        const int x2 = (int)t2 - x3 * g.N2;
        const int rp = (x1 + x2 + x3 + parity) & 1;            // x0 = 2*hx0 + rp
        int nf[4], nb[4];
        nf[0] = rp ? (hx0 + 1 == g.Nh0 ? i - (g.Nh0 - 1) : i + 1) : i;
        nb[0] = rp ? i : (hx0 == 0 ? i + (g.Nh0 - 1) : i - 1);
        nf[1] = x1 + 1 == g.N1 ? i - (g.N1 - 1) * g.s1 : i + g.s1;
        nb[1] = x1 == 0 ? i + (g.N1 - 1) * g.s1 : i - g.s1;
        nf[2] = x2 + 1 == g.N2 ? i - (g.N2 - 1) * g.s2 : i + g.s2;
        nb[2] = x2 == 0 ? i + (g.N2 - 1) * g.s2 : i - g.s2;
        nf[3] = x3 + 1 == g.N3 ? i - (g.N3 - 1) * g.s3 : i + g.s3;
        nb[3] = x3 == 0 ? i + (g.N3 - 1) * g.s3 : i - g.s3;
        // 1/2 * eta_mu(x) (readings R2, R3); boundary sign on the x3 hops (reading R4)
        T cf[4], cb[4];
        const T h = (T)0.5;
        cf[0] = h;
        cf[1] = rp ? -h : h;
        cf[2] = ((rp + x1) & 1) ? -h : h;
        cf[3] = ((rp + x1 + x2) & 1) ? -h : h;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) cb[mu] = -cf[mu];
        if (g.ap) {
            if (x3 == g.N3 - 1) cf[3] = -cf[3];
            if (x3 == 0) cb[3] = -cb[3];
        }
        // ---- a3, a4: 8 hops -----------------------------------------------------------------
        Cx<T> acc[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[c] = cx<T>((T)0, (T)0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            {
                Su3<T> u = load_link<T, LAYOUT, RECON12, POLICY>(links, parity, mu, (size_t)g.Ls, (size_t)i, pol);
                Cx<T> p[3];
                if (HALO && mu == 3 && nf[3] >= i_end) {
                    T cr, ci;
                    phase_coef<T, BF>(bf, (size_t)(parity * 4 + 3) * Vh + i, cf[3], (T)1, &cr, &ci);
                    load_vec_cg<T, LAYOUT>((const T *)pdp->land_self[1 - parity][1], (size_t)g.s3, (size_t)(nf[3] - i_end), cr, ci, p);
                }
                else if (BF == 1) load_vec_phase<T, LAYOUT, POLICY>(in, Vh, (size_t)nf[mu], cf[mu], __ldcs(bf + (size_t)(parity * 4 + mu) * Vh + i), p, pol);
                else if (BF == 2) load_vec_unit<T, LAYOUT, POLICY>(in, Vh, (size_t)nf[mu], cf[mu], (T)1, bf, (size_t)(parity * 4 + mu) * Vh + i, p, pol);
                else load_vec<T, LAYOUT, POLICY>(in, Vh, (size_t)nf[mu], cf[mu], p, pol);
                mv_acc<T>(acc, u, p);
            }
            {
                Su3<T> u = load_link<T, LAYOUT, RECON12, POLICY>(links, 1 - parity, mu, (size_t)g.Ls, (size_t)nb[mu], pol);
                Cx<T> p[3];
                if (HALO && mu == 3 && nb[3] < i_begin) {
                    T cr, ci;
                    phase_coef<T, BF>(bf, (size_t)((1 - parity) * 4 + 3) * Vh + nb[3], cb[3], (T)-1, &cr, &ci);
                    load_vec_cg<T, LAYOUT>((const T *)pdp->land_self[1 - parity][0], (size_t)g.s3, (size_t)(nb[3] - (i_begin - g.s3)), cr, ci, p);
                }
                else if (BF == 1) load_vec_phase<T, LAYOUT, POLICY>(in, Vh, (size_t)nb[mu], cb[mu], -__ldcs(bf + (size_t)((1 - parity) * 4 + mu) * Vh + nb[mu]), p, pol);
                else if (BF == 2) load_vec_unit<T, LAYOUT, POLICY>(in, Vh, (size_t)nb[mu], cb[mu], (T)-1, bf, (size_t)((1 - parity) * 4 + mu) * Vh + nb[mu], p, pol);
                else load_vec<T, LAYOUT, POLICY>(in, Vh, (size_t)nb[mu], cb[mu], p, pol);
                mvdag_acc<T>(acc, u, p);
            }
        }
        // ---- a5: epilogue ------------------------------------------------------------------
        if (MODE >= 1) {
            const T cm = (T)coef;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                Cx<T> x = ld_cx<T, LAYOUT, 0, POLICY>(xin, (size_t)c, Vh, (size_t)i, pol);
                acc[c] = cx<T>(fma(cm, x.re, -acc[c].re), fma(cm, x.im, -acc[c].im));
                if (MODE == 2) dot += (double)x.re * (double)acc[c].re + (double)x.im * (double)acc[c].im;
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) st_cx<T, LAYOUT, POLICY>(out, (size_t)c, Vh, (size_t)i, acc[c], pol);
        if (HALO && push_out) {
            // the face push fused into the producer: the owned boundary slices of `out` (times the boundary sign)
            // go straight into the neighbours' landing buffers; the next Dslash raises the flags
            if (i < i_begin + g.s3) {
                const T sg = (T)pdp->sign_down;
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    st_cx<T, LAYOUT, 0>((T *)pdp->land_down[parity], (size_t)c, (size_t)g.s3, (size_t)(i - i_begin), cx<T>(sg * acc[c].re, sg * acc[c].im), pol);
            }
            if (i >= i_end - g.s3) {
                const T sg = (T)pdp->sign_up;
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    st_cx<T, LAYOUT, 0>((T *)pdp->land_up[parity], (size_t)c, (size_t)g.s3, (size_t)(i - (i_end - g.s3)), cx<T>(sg * acc[c].re, sg * acc[c].im), pol);
            }
        }
    }
    }
    if (MODE == 2) {
        if (HALO) {       // slab mode, peer transport: per-CTA partials as on one GPU; K1's CTA 0 adds them up and publishes
            const double b = block_sum(dot);
            if (threadIdx.x == 0) partials[bx] = b;
            if (blockIdx.x == 0 && threadIdx.x == 0) peer_bump_red(*pdp, 0);
        } else if (st->comm) {   // slab mode: the caller all-reduces the LOCAL total (lqcd_set_slab)
            double total;
            if (grid_sum_last(dot, partials, &st->ticket, &total)) st->sum[0] = total;
        } else {          // the next kernel (K1) adds the partials up itself: no fence, no ticket, no tail
            const double b = block_sum(dot);
            if (threadIdx.x == 0) partials[blockIdx.x] = b;
        }
    }
}

template <typename T, int LAYOUT, int RECON12, int MODE>
static void launch_t(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                     const void *xin, double coef, int gate, int i_begin, int i_end, int halo_in, int push_out)
{
    int block = ctx->dslash_block > 256 ? 256 : ctx->dslash_block;
    int tiles = (i_end - i_begin + block - 1) / block;
    if (tiles < 1) tiles = 1;
    if (ctx->dslash_persist > 0 && tiles > ctx->num_sms * ctx->dslash_persist) tiles = ctx->num_sms * ctx->dslash_persist;
    dim3 grid(tiles);
    ctx->last_dslash_grid = tiles;
    int minb = ctx->dslash_minblocks;
    if (minb == 0) minb = sizeof(T) == 8 ? 2 : 4;   // profiles/experiments_r1b.md section 9
#define GO1(MB, P, B) GO2(MB, P, B, 0)
#define GO2(MB, P, B, H) launch_k(ctx, dslash_kernel<T, LAYOUT, RECON12, MODE, MB, P, B, H>, grid, dim3(block), \
        ctx->g, parity, (T *)out, (const T *)in, (const T *)links, (const T *)xin, coef, ctx->d_state, ctx->d_partials, gate, i_begin, i_end, \
        (const T *)ctx->backfield, (const PeerDev *)ctx->d_peer, push_out)
#define GO(MB) do { if (ctx->l2_hints) GO1(MB, 1, 0); else GO1(MB, 0, 0); } while (0)
    // peer transport: the per-precision default variant, faces read from the landing buffers (halo_in)
    // (DEF_MB is a compile-time constant so that only the variant a precision can launch is instantiated)
    constexpr int DEF_MB = sizeof(T) == 8 ? 2 : 4;
    if (halo_in) {
        const int b = ctx->backfield ? 1 + ctx->backfield_format : 0;
        if (b == 0) GO2(DEF_MB, 0, 0, 1); else if (b == 1) GO2(DEF_MB, 0, 1, 1); else GO2(DEF_MB, 0, 2, 1);
    } else
    // with a backfield: the per-precision default variant only (the tuning options dslash_minblocks and
    // l2_hints select nothing there)
    if (ctx->backfield && ctx->backfield_format == 0) GO1(DEF_MB, 0, 1);
    else if (ctx->backfield) GO1(DEF_MB, 0, 2);
    else if (minb <= 2) GO(2); else if (minb == 3) GO(3); else GO(4);
#undef GO
#undef GO1
#undef GO2
}

template <typename T, int LAYOUT>
static void launch_tl(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                      const void *xin, double coef, int mode, int gate, int i_begin, int i_end, int halo_in, int push_out)
{
#define GO(R, M) launch_t<T, LAYOUT, R, M>(ctx, parity, out, in, links, xin, coef, gate, i_begin, i_end, halo_in, push_out)
    if (ctx->recon == LQCD_RECON_12) { if (mode == 0) GO(1, 0); else if (mode == 1) GO(1, 1); else GO(1, 2); }
    else { if (mode == 0) GO(0, 0); else if (mode == 1) GO(0, 1); else GO(0, 2); }
#undef GO
}

int launch_dslash(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                  const void *xpay_in, double coef, int dot_mode, int gate, int x3_lo, int x3_hi, int push_out)
{
    int mode = xpay_in ? (dot_mode ? 2 : 1) : 0;
    // peer transport: a Dslash over the context's owned slices reads the faces the neighbours pushed; an explicit
    // slice range (lqcd_dslash_slices) reads the vector's own ghost slices as before
    const int halo_in = ctx->peer_on && x3_lo < 0;
    if (x3_lo < 0) { x3_lo = ctx->x3_lo; x3_hi = ctx->x3_hi; }      // the context's interior slices
    const int i_begin = x3_lo * ctx->g.s3, i_end = x3_hi * ctx->g.s3;
    if (ctx->prec == LQCD_F64) {
        if (ctx->layout == 0) launch_tl<double, 0>(ctx, parity, out, in, links, xpay_in, coef, mode, gate, i_begin, i_end, halo_in, halo_in ? push_out : 0);
        else launch_tl<double, 1>(ctx, parity, out, in, links, xpay_in, coef, mode, gate, i_begin, i_end, halo_in, halo_in ? push_out : 0);
    } else {
        if (ctx->layout == 0) launch_tl<float, 0>(ctx, parity, out, in, links, xpay_in, coef, mode, gate, i_begin, i_end, halo_in, halo_in ? push_out : 0);
        else launch_tl<float, 1>(ctx, parity, out, in, links, xpay_in, coef, mode, gate, i_begin, i_end, halo_in, halo_in ? push_out : 0);
    }
    return lqcd_check_cuda(ctx, cudaGetLastError(), "dslash");
}
