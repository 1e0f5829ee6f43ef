// force.cu -- fermion-force outer products (the step after
// the multi-shift solve, "a large fraction of the execution time is spent in ... deo and doe").
// The paper gives no formula (it follows its ref. 33); reading R21 of DESIGN.md:
//
//   S = phi^dagger r(A) phi,  r(A) = c0 + sum_i c_i (A + sigma_i)^-1,  A = m^2 - D_eo D_oe   (Eq. 3, 6, 8)
//   x_i = (A + sigma_i)^-1 phi (even sites), y_i = D_oe x_i (odd sites), w_i = x_i | y_i by parity
//   F_mu(x) = TA[ U_mu(x) Q_mu(x) ],   dS/d eps = 2 Re Tr[i T F_mu(x)]  for U_mu(x) -> exp(i eps T) U_mu(x)
//   Q_mu(x) = 1/2 eta_mu(x) s+_mu(x) (-1)^{p(x)} sum_i c_i w_i(x+mu) w_i(x)^dagger
//   TA[M]   = (M - M^dagger)/2 - Tr(M - M^dagger)/6
//
// One thread per site, the four directions in turn: per direction the n outer products are
// accumulated in registers (the site's own n vectors are re-read from L1 for each direction), then
// U_mu(x) is streamed in once, multiplied, projected and the 3x3 result stored.  HBM-bound like the
// Dslash: per full-lattice site 576 B of links + 48 n B of vectors (each w_i once; the 4 neighbour
// reads hit L1/L2) + 576 B of force written; the n Dslash applications that produce the y_i come on top.
#include "su3.cuh"

void *ws_vec(lqcd_ctx *ctx, int k);   // api.cu

struct ForceVecs {
    const void *self[LQCD_MAX_SHIFTS];   // w_i on the sites of the launch's parity
    const void *nbr[LQCD_MAX_SHIFTS];    // w_i on the other parity
    double coef[LQCD_MAX_SHIFTS];        // c_i (-1)^parity
    int n;
};

// STAGE = 1: the site's own n vectors are read from global memory ONCE into the thread's private
// column of dynamic shared memory (n * 6 reals * 128 threads <= 48 KB) and re-read from there for each
// direction; ncu had shown the four re-reads missing L1 (hit rate 0.8 %) and costing +33 % DRAM reads.
template <typename T, int LAYOUT, int RECON12, int STAGE>
__global__ void __launch_bounds__(128, 5) force_kernel(const Geom g, const int parity, T *__restrict__ force,
                                                    const T *__restrict__ links, const ForceVecs fv,
                                                    const T *__restrict__ bf, const int bf_fmt, const int i_begin, const int i_end)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *const own = reinterpret_cast<T *>(smem_raw);      // own[(s*6 + k)*128 + tid]
    pdl_wait();
    pdl_trigger();
    // sites [i_begin, i_end): the whole parity, or the owned x3 slices of a slab (the forward x3 neighbours of the top
    // owned slice are then read from the vectors' ghost slice, which the caller's halo exchange has filled)
    const int i = i_begin + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= i_end) return;
    const size_t Vh = (size_t)g.Vh;
    const L2Pol pol = {0, 0};
    // site decode and forward neighbours as in dslash.cu (Eq. 9)
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    const int hx0 = i - (int)t * g.Nh0;
    uint32_t t2 = fd_div(t, g.dN1);
    const int x1 = (int)t - (int)t2 * g.N1;
    const int x3 = (int)fd_div(t2, g.dN2);
    const int x2 = (int)t2 - x3 * g.N2;
    const int rp = (x1 + x2 + x3 + parity) & 1;
    int nf[4];
    nf[0] = rp ? (hx0 + 1 == g.Nh0 ? i - (g.Nh0 - 1) : i + 1) : i;
    nf[1] = x1 + 1 == g.N1 ? i - (g.N1 - 1) * g.s1 : i + g.s1;
    nf[2] = x2 + 1 == g.N2 ? i - (g.N2 - 1) * g.s2 : i + g.s2;
    nf[3] = x3 + 1 == g.N3 ? i - (g.N3 - 1) * g.s3 : i + g.s3;
    T e[4];
    const T h = (T)0.5;
    e[0] = h;
    e[1] = rp ? -h : h;
    e[2] = ((rp + x1) & 1) ? -h : h;
    e[3] = ((rp + x1 + x2) & 1) ? -h : h;
    if (g.ap && x3 == g.N3 - 1) e[3] = -e[3];

    if (STAGE) {
        for (int s = 0; s < fv.n; ++s) {
            Cx<T> ws[3];
            load_vec<T, LAYOUT, 0>((const T *)fv.self[s], Vh, (size_t)i, (T)1, ws, pol);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                own[(s * 6 + 2 * c) * 128 + threadIdx.x] = ws[c].re;
                own[(s * 6 + 2 * c + 1) * 128 + threadIdx.x] = ws[c].im;
            }
        }
    }
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        Cx<T> Q[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) Q[a][b] = cx<T>((T)0, (T)0);
        for (int s = 0; s < fv.n; ++s) {
            Cx<T> ws[3], wn[3];
            if (STAGE) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    ws[c] = cx<T>(own[(s * 6 + 2 * c) * 128 + threadIdx.x], own[(s * 6 + 2 * c + 1) * 128 + threadIdx.x]);
            } else load_vec<T, LAYOUT, 0>((const T *)fv.self[s], Vh, (size_t)i, (T)1, ws, pol);
            load_vec<T, LAYOUT, 0>((const T *)fv.nbr[s], Vh, (size_t)nf[mu], (T)fv.coef[s], wn, pol);
            // Q[a][b] += c w(x+mu)[a] conj(w(x)[b])
            // (requesting the neighbour vectors of 2 / 4 / 8 shifts together was tried in round 2 and is slower at
            // every batch size: profiles/sweep_r2.md section 5)
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    Q[a][b].re = fma(wn[a].re, ws[b].re, Q[a][b].re);
                    Q[a][b].re = fma(wn[a].im, ws[b].im, Q[a][b].re);
                    Q[a][b].im = fma(wn[a].im, ws[b].re, Q[a][b].im);
                    Q[a][b].im = fma(-wn[a].re, ws[b].im, Q[a][b].im);
                }
        }
        const Su3<T> u = load_link<T, LAYOUT, RECON12, 0>(links, parity, mu, (size_t)g.Ls, (size_t)i, pol);
        // backfield (reading R6): the link of D is e^{i theta} U, and so is the link of the force
        T pr = e[mu], pi = (T)0;
        if (bf) {
            T sn, cs;
            const size_t k = (size_t)(parity * 4 + mu) * Vh + i;
            if (bf_fmt == 0) sincos_t(__ldcs(bf + k), &sn, &cs);
            else { cs = __ldcs(bf + 2 * k); sn = __ldcs(bf + 2 * k + 1); }
            pr = e[mu] * cs; pi = e[mu] * sn;
        }
        Cx<T> M[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                T re = 0, im = 0;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    re = fma(u.e[a][k].re, Q[k][b].re, re);
                    re = fma(-u.e[a][k].im, Q[k][b].im, re);
                    im = fma(u.e[a][k].re, Q[k][b].im, im);
                    im = fma(u.e[a][k].im, Q[k][b].re, im);
                }
                M[a][b] = cx<T>(pr * re - pi * im, pr * im + pi * re);
            }
        // TA[M]: Tr(M - M^dagger) = 2 i sum_a Im M_aa
        const T tr3 = (M[0][0].im + M[1][1].im + M[2][2].im) / (T)3;
        // F is traceless anti-Hermitian: 8 reals (the paper's tamat_soa).  Planes per
        // (parity, mu): F01, F02, F12 and (Im F00, Im F11); lqcd_unpack_tamat rebuilds the 3x3 matrix.
        const size_t pl = (size_t)(parity * 4 + mu) * 4;
        st_cx<T, LAYOUT, 0>(force, pl + 0, Vh, (size_t)i, cx<T>((T)0.5 * (M[0][1].re - M[1][0].re), (T)0.5 * (M[0][1].im + M[1][0].im)), pol);
        st_cx<T, LAYOUT, 0>(force, pl + 1, Vh, (size_t)i, cx<T>((T)0.5 * (M[0][2].re - M[2][0].re), (T)0.5 * (M[0][2].im + M[2][0].im)), pol);
        st_cx<T, LAYOUT, 0>(force, pl + 2, Vh, (size_t)i, cx<T>((T)0.5 * (M[1][2].re - M[2][1].re), (T)0.5 * (M[1][2].im + M[2][1].im)), pol);
        st_cx<T, LAYOUT, 0>(force, pl + 3, Vh, (size_t)i, cx<T>(M[0][0].im - tr3, M[1][1].im - tr3), pol);
    }
}

// native force field (planes ((parity*4 + mu)*3 + row)*3 + col of Vh sites) -> canonical c128 [V][4][3][3]
template <typename T, int LAYOUT>
__global__ void unpack_force_kernel(Geom g, double2 *__restrict__ canon, const T *__restrict__ native)
{
    pdl_wait();
    pdl_trigger();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int par = blockIdx.y;
    if (i >= g.Vh) return;
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    uint32_t t2 = fd_div(t, g.dN1);
    const int x1 = (int)t - (int)t2 * g.N1;
    const int x3 = (int)fd_div(t2, g.dN2);
    const int x2 = (int)t2 - x3 * g.N2;
    const size_t lex = 2 * (size_t)i + ((x1 + x2 + x3 + par) & 1);
    for (int mu = 0; mu < 4; ++mu)
        for (int k = 0; k < 9; ++k) {
            Cx<T> z = ld_cx<T, LAYOUT, 0, 0>(native, (size_t)((par * 4 + mu) * 9 + k), (size_t)g.Vh, (size_t)i, L2Pol());
            canon[(lex * 4 + mu) * 9 + k] = make_double2((double)z.re, (double)z.im);
        }
}

// native tamat field (4 complex planes per (parity, mu)) -> canonical c128 [V][4][3][3]
template <typename T, int LAYOUT>
__global__ void unpack_tamat_kernel(Geom g, double2 *__restrict__ canon, const T *__restrict__ native)
{
    pdl_wait();
    pdl_trigger();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int par = blockIdx.y;
    if (i >= g.Vh) return;
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    uint32_t t2 = fd_div(t, g.dN1);
    const int x1 = (int)t - (int)t2 * g.N1;
    const int x3 = (int)fd_div(t2, g.dN2);
    const int x2 = (int)t2 - x3 * g.N2;
    const size_t lex = 2 * (size_t)i + ((x1 + x2 + x3 + par) & 1);
    for (int mu = 0; mu < 4; ++mu) {
        Cx<T> z[4];
        for (int k = 0; k < 4; ++k) z[k] = ld_cx<T, LAYOUT, 0, 0>(native, (size_t)((par * 4 + mu) * 4 + k), (size_t)g.Vh, (size_t)i, L2Pol());
        double2 *f = canon + (lex * 4 + mu) * 9;
        const double a = (double)z[3].re, b = (double)z[3].im;
        f[0] = make_double2(0.0, a);
        f[1] = make_double2((double)z[0].re, (double)z[0].im);
        f[2] = make_double2((double)z[1].re, (double)z[1].im);
        f[3] = make_double2(-(double)z[0].re, (double)z[0].im);      // F10 = -conj(F01)
        f[4] = make_double2(0.0, b);
        f[5] = make_double2((double)z[2].re, (double)z[2].im);
        f[6] = make_double2(-(double)z[1].re, (double)z[1].im);
        f[7] = make_double2(-(double)z[2].re, (double)z[2].im);
        f[8] = make_double2(0.0, -(a + b));
    }
}

extern "C" size_t lqcd_tamat_bytes(const lqcd_ctx *ctx)
{
    return ctx ? (size_t)ctx->g.Vh * 2 * 4 * 4 * 2 * elem_size(ctx) : 0;
}

extern "C" int lqcd_unpack_tamat(lqcd_ctx *ctx, void *canonical_dev, const void *native)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!canonical_dev || !native) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_unpack_tamat: null pointer");
    dim3 grid((ctx->g.Vh + 127) / 128, 2), block(128);
    if (ctx->prec == LQCD_F64) {
        if (ctx->layout == 0) launch_k(ctx, unpack_tamat_kernel<double, 0>, grid, block, ctx->g, (double2 *)canonical_dev, (const double *)native);
        else launch_k(ctx, unpack_tamat_kernel<double, 1>, grid, block, ctx->g, (double2 *)canonical_dev, (const double *)native);
    } else {
        if (ctx->layout == 0) launch_k(ctx, unpack_tamat_kernel<float, 0>, grid, block, ctx->g, (double2 *)canonical_dev, (const float *)native);
        else launch_k(ctx, unpack_tamat_kernel<float, 1>, grid, block, ctx->g, (double2 *)canonical_dev, (const float *)native);
    }
    return lqcd_check_cuda(ctx, cudaGetLastError(), "unpack_tamat");
}

extern "C" size_t lqcd_force_bytes(const lqcd_ctx *ctx)
{
    return ctx ? (size_t)ctx->g.Vh * 2 * 4 * 9 * 2 * elem_size(ctx) : 0;
}

template <typename T, int LAYOUT>
static void launch_force_tl(lqcd_ctx *ctx, int parity, void *force, const void *links, const ForceVecs &fv)
{
    const int i_begin = ctx->x3_lo * ctx->g.s3, i_end = ctx->x3_hi * ctx->g.s3;
    dim3 grid((i_end - i_begin + 127) / 128), block(128);
    const size_t smem = (size_t)fv.n * 6 * 128 * sizeof(T);
    // measured at 32^4 (profiles/experiments_r1b.md section 7): fp64 -3 %, fp32 +20 % (the carve-out costs L1)
    if (smem <= 48 * 1024 && ctx->force_stage && sizeof(T) == 8) {
        if (ctx->recon == LQCD_RECON_12) launch_k_smem(ctx, force_kernel<T, LAYOUT, 1, 1>, grid, block, smem, ctx->g, parity, (T *)force, (const T *)links, fv, (const T *)ctx->backfield, ctx->backfield_format, i_begin, i_end);
        else launch_k_smem(ctx, force_kernel<T, LAYOUT, 0, 1>, grid, block, smem, ctx->g, parity, (T *)force, (const T *)links, fv, (const T *)ctx->backfield, ctx->backfield_format, i_begin, i_end);
    } else {
        if (ctx->recon == LQCD_RECON_12) launch_k(ctx, force_kernel<T, LAYOUT, 1, 0>, grid, block, ctx->g, parity, (T *)force, (const T *)links, fv, (const T *)ctx->backfield, ctx->backfield_format, i_begin, i_end);
        else launch_k(ctx, force_kernel<T, LAYOUT, 0, 0>, grid, block, ctx->g, parity, (T *)force, (const T *)links, fv, (const T *)ctx->backfield, ctx->backfield_format, i_begin, i_end);
    }
}

extern "C" int lqcd_fermion_force(lqcd_ctx *ctx, int nshift, const double *coeffs, void *const *xs_e,
                                  const void *links, void *force)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return lqcd_fail(ctx, LQCD_ERR_ARG, "nshift %d not in [1,%d]", nshift, LQCD_MAX_SHIFTS);
    if (!coeffs || !xs_e || !links || !force) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_fermion_force: null pointer");
    for (int i = 0; i < nshift; ++i) {
        if (!xs_e[i]) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_fermion_force: solution %d is null", i);
        if (coeffs[i] != coeffs[i]) return lqcd_fail(ctx, LQCD_ERR_ARG, "coefficient %d is NaN", i);
    }
    const bool slab = ctx->halo_fn || ctx->peer_on;
    if (!slab && (ctx->x3_lo != 0 || ctx->x3_hi != ctx->g.N3))
        return lqcd_fail(ctx, LQCD_ERR_UNSUPPORTED, "lqcd_fermion_force: a slab context needs a transport (lqcd_set_slab hooks or lqcd_peer_connect)");
    if (!ctx->ws) return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "no workspace set");
    if (ctx->ws_bytes < lqcd_workspace_bytes(ctx, nshift))
        return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "workspace %zu bytes < %zu needed for %d shifts", ctx->ws_bytes, lqcd_workspace_bytes(ctx, nshift), nshift);
    // y_i = D_oe x_i into the workspace slots the solver uses for its p_i.  In slab mode the solutions live on the local
    // parity `par` (the paper's even sites), y_i on the other one, and the force kernel reads the forward x3
    // neighbours of the top owned slice from the vectors' ghost slices: both x_i and y_i get their ghosts filled.
    const int par = ctx->solve_parity;
    auto ghosts = [&](void *v, int parity) -> int {
        if (ctx->peer_on) { int e = launch_peer_push(ctx, v, parity, 0); return e ? e : launch_peer_pull(ctx, v, parity); }
        if (ctx->halo_fn && ctx->halo_fn(ctx->comm_user, v, parity)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "halo hook failed");
        return LQCD_OK;
    };
    ForceVecs fx, fy;             // launches on the sites of parity par / 1 - par
    memset(&fx, 0, sizeof(fx));
    memset(&fy, 0, sizeof(fy));
    fx.n = fy.n = nshift;
    // plain context: all y_i from the block Dslash, which loads every link once per block of right-hand sides instead
    // of once per shift (dslash_multi.cu); slab contexts and a backfield keep one Dslash per shift
    const bool block = !slab && !ctx->backfield && ctx->force_block >= 2 && nshift >= 2;
    if (block) {
        void *ys[LQCD_MAX_SHIFTS];
        for (int i = 0; i < nshift; ++i) ys[i] = ws_vec(ctx, 4 + i);
        if ((rc = launch_dslash_multi(ctx, 1 - par, nshift, ys, (const void *const *)xs_e, links, ctx->force_block))) return rc;
    }
    for (int i = 0; i < nshift; ++i) {
        void *y = ws_vec(ctx, 4 + i);
        if (!block) {
            if ((rc = ghosts(xs_e[i], par))) return rc;
            if ((rc = launch_dslash(ctx, 1 - par, y, xs_e[i], links, NULL, 0.0, 0, 0))) return rc;
            if (slab && (rc = ghosts(y, 1 - par))) return rc;
        }
        fx.self[i] = xs_e[i]; fx.nbr[i] = y; fx.coef[i] = coeffs[i];        // x even: + c_i y_i(x+mu) x_i(x)^dagger
        fy.self[i] = y; fy.nbr[i] = xs_e[i]; fy.coef[i] = -coeffs[i];       // x odd:  - c_i x_i(x+mu) y_i(x)^dagger
    }
    for (int k = 0; k < 2; ++k) {
        const int lp = k ? 1 - par : par;
        const ForceVecs &fv = k ? fy : fx;
        if (ctx->prec == LQCD_F64) {
            if (ctx->layout == 0) launch_force_tl<double, 0>(ctx, lp, force, links, fv); else launch_force_tl<double, 1>(ctx, lp, force, links, fv);
        } else {
            if (ctx->layout == 0) launch_force_tl<float, 0>(ctx, lp, force, links, fv); else launch_force_tl<float, 1>(ctx, lp, force, links, fv);
        }
    }
    return lqcd_check_cuda(ctx, cudaGetLastError(), "fermion force");
}

extern "C" int lqcd_unpack_force(lqcd_ctx *ctx, void *canonical_dev, const void *native)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!canonical_dev || !native) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_unpack_force: null pointer");
    dim3 grid((ctx->g.Vh + 127) / 128, 2), block(128);
    if (ctx->prec == LQCD_F64) {
        if (ctx->layout == 0) launch_k(ctx, unpack_force_kernel<double, 0>, grid, block, ctx->g, (double2 *)canonical_dev, (const double *)native);
        else launch_k(ctx, unpack_force_kernel<double, 1>, grid, block, ctx->g, (double2 *)canonical_dev, (const double *)native);
    } else {
        if (ctx->layout == 0) launch_k(ctx, unpack_force_kernel<float, 0>, grid, block, ctx->g, (double2 *)canonical_dev, (const float *)native);
        else launch_k(ctx, unpack_force_kernel<float, 1>, grid, block, ctx->g, (double2 *)canonical_dev, (const float *)native);
    }
    return lqcd_check_cuda(ctx, cudaGetLastError(), "unpack_force");
}
