// dslash_multi.cu -- the even/odd staggered Dirac operator applied to several right-hand sides at once (a "block"
// Dslash): out_r = D in_r for r = 0..NRHS-1 on the sites of one parity (Eq. 7; same stencil,
// phases and boundary sign as dslash.cu, readings R1-R5, R8).
//
// Why: after the multi-shift solve the fermion force needs y_i = D_oe x_i for every shift ("a large
// fraction of the execution time is spent in ... deo and doe"; reading R21).  One Dslash per shift reads the link
// field once per shift: 1248 B per odd site and shift in fp64, 1152 of them links.  The links do not depend on the
// right-hand side: here a thread loads each of its 8 links ONCE, rebuilds the third row once (2-row storage), and
// multiplies NRHS neighbour vectors by it.  Algorithmic bytes per site: 1152 + 96 NRHS (fp64, 18-real) instead of
// 1248 NRHS -- for the 8 shifts of the rational approximation 1920 (one launch of 8) or 3072 (two launches of 4)
// instead of 9984.  Still bound by HBM, not by FP64: 570 flop per site and right-hand side against >= 240 B.
//
// Scope: the whole parity of a plain context (no backfield, no slab / peer transport: lqcd_fermion_force keeps the
// one-vector kernel there).  Per right-hand side the arithmetic is the one of dslash_kernel<MODE 0> in the same
// order, so the results are bit-identical to NRHS single applications.
#include "su3.cuh"

template <int NRHS> struct MultiVecs { void *out[NRHS]; const void *in[NRHS]; };

template <typename T, int LAYOUT, int RECON12, int NRHS, int MINB>
__global__ void __launch_bounds__(128, MINB)
dslash_multi_kernel(const Geom g, const int parity, const MultiVecs<NRHS> v, const T *__restrict__ links)
{
    pdl_wait();
    pdl_trigger();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    const L2Pol pol = {0, 0};
    const size_t Vh = (size_t)g.Vh;
    // ---- a2: site decode (Eq. 9), neighbours, phases: as in dslash_kernel --------------------------------
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
    // ---- a3, a4: 8 hops, each link loaded once for all right-hand sides ----------------------------------
    Cx<T> acc[NRHS][3];
#pragma unroll
    for (int r = 0; r < NRHS; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[r][c] = cx<T>((T)0, (T)0);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        {
            const Su3<T> u = load_link<T, LAYOUT, RECON12, 0>(links, parity, mu, (size_t)g.Ls, (size_t)i, pol);
#pragma unroll
            for (int r = 0; r < NRHS; ++r) {
                Cx<T> p[3];
                load_vec<T, LAYOUT, 0>((const T *)v.in[r], Vh, (size_t)nf[mu], cf[mu], p, pol);
                mv_acc<T>(acc[r], u, p);
            }
        }
        {
            const Su3<T> u = load_link<T, LAYOUT, RECON12, 0>(links, 1 - parity, mu, (size_t)g.Ls, (size_t)nb[mu], pol);
#pragma unroll
            for (int r = 0; r < NRHS; ++r) {
                Cx<T> p[3];
                load_vec<T, LAYOUT, 0>((const T *)v.in[r], Vh, (size_t)nb[mu], cb[mu], p, pol);
                mvdag_acc<T>(acc[r], u, p);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < NRHS; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) st_cx<T, LAYOUT, 0>((T *)v.out[r], (size_t)c, Vh, (size_t)i, acc[r][c], pol);
}

template <typename T, int LAYOUT, int RECON12, int NRHS, int MINB>
static void launch_n(lqcd_ctx *ctx, int parity, void *const *outs, const void *const *ins, const void *links)
{
    MultiVecs<NRHS> v;
    for (int r = 0; r < NRHS; ++r) { v.out[r] = outs[r]; v.in[r] = ins[r]; }
    launch_k(ctx, dslash_multi_kernel<T, LAYOUT, RECON12, NRHS, MINB>, dim3((ctx->g.Vh + 127) / 128), dim3(128), ctx->g, parity, v, (const T *)links);
}

template <typename T, int LAYOUT, int RECON12>
static void launch_blocks(lqcd_ctx *ctx, int parity, int n, void *const *outs, const void *const *ins, const void *links, int blk)
{
    // fp64: 4 right-hand sides = 24 accumulators + 18 link + 6 vector doubles fit 168 registers (3 CTAs of 128 per SM);
    // 8 need the full 255 (2 CTAs per SM).  fp32 values take one register each.
    constexpr int MB4 = sizeof(T) == 8 ? 3 : 4, MB8 = sizeof(T) == 8 ? 2 : 3;
    int k = 0;
    if (blk >= 8) for (; k + 8 <= n; k += 8) launch_n<T, LAYOUT, RECON12, 8, MB8>(ctx, parity, outs + k, ins + k, links);
    for (; k + 4 <= n; k += 4) launch_n<T, LAYOUT, RECON12, 4, MB4>(ctx, parity, outs + k, ins + k, links);
    for (; k + 2 <= n; k += 2) launch_n<T, LAYOUT, RECON12, 2, MB4>(ctx, parity, outs + k, ins + k, links);
    for (; k < n; ++k) launch_n<T, LAYOUT, RECON12, 1, MB4>(ctx, parity, outs + k, ins + k, links);
}

// outs[r] = D ins[r] on the sites of `parity`, r = 0..n-1, in blocks of up to `blk` (4 or 8) right-hand sides per launch.
// Plain contexts only (the caller checks): whole parity, no backfield, no transport.
int launch_dslash_multi(lqcd_ctx *ctx, int parity, int n, void *const *outs, const void *const *ins, const void *links, int blk)
{
#define GO(T, L) do { if (ctx->recon == LQCD_RECON_12) launch_blocks<T, L, 1>(ctx, parity, n, outs, ins, links, blk); \
                      else launch_blocks<T, L, 0>(ctx, parity, n, outs, ins, links, blk); } while (0)
    if (ctx->prec == LQCD_F64) { if (ctx->layout == 0) GO(double, 0); else GO(double, 1); }
    else { if (ctx->layout == 0) GO(float, 0); else GO(float, 1); }
#undef GO
    return lqcd_check_cuda(ctx, cudaGetLastError(), "block dslash");
}
