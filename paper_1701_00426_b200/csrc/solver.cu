// solver.cu -- CG and multi-shift CG on A = m^2 - D_eo D_oe (Eq. 8; the
// "multishift inverter routine" of PAPER.md:313 for Eq. 6), readings R10-R14, R16.
//
// Steps a5-a8 of SURVEY.md section 8(a).  Per iteration, on one stream, with no host round trip:
//   K_A  tmp_o = D_oe p                                              (dslash.cu)
//   K_B  q = (m^2 + sigma_min) p - D_eo tmp_o ;  Re<p,q>  -> alpha, zeta_i^new, alpha_i
//   K1   r -= alpha q ;  <r,r>                             -> beta, beta_i, freeze flags
//   K2   x_i += alpha_i p_i ;  p_i = zeta_i^new r + beta_i p_i ;  p = r + beta p   (one pass)
// The paper's "zaxpy-like functions" and dot products are these two fused
// kernels; the scalars live in a device struct and are produced by the last CTA of each
// reduction.  The host only polls a `done` word every poll_chunk iterations.
//
// The vector kernels are layout-agnostic: every update is (real scalar) x (vector), so they run
// over the 6*Vh reals of a half-lattice vector as a flat array with 16-byte loads.
#include <stdlib.h>

#include "peer.cuh"
#include "reduce.cuh"

void *ws_vec(lqcd_ctx *ctx, int k);   // api.cu

template <typename T> struct Pack;            // 16-byte packet of reals
template <> struct Pack<double> { typedef double2 type; enum { N = 2 }; };
template <> struct Pack<float> { typedef float4 type; enum { N = 4 }; };

template <typename T> __device__ __forceinline__ void unpack(const double2 &v, T *a) { a[0] = v.x; a[1] = v.y; }
template <typename T> __device__ __forceinline__ void unpack(const float4 &v, T *a) { a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
__device__ __forceinline__ double2 repack(const double *a) { return make_double2(a[0], a[1]); }
__device__ __forceinline__ float4 repack(const float *a) { return make_float4(a[0], a[1], a[2], a[3]); }

// 16-byte vector loads / stores of the flat kernels; POLICY 1 adds L2::evict_last so that the
// CG vectors stay L2-resident between kernels (common.cuh).  Plain (coherent) loads: these
// kernels read and write the same buffers.
template <int POLICY> __device__ __forceinline__ double2 ldv(const double2 *p, uint64_t pol)
{
    if (POLICY == 0) return *p;
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
template <int POLICY> __device__ __forceinline__ float4 ldv(const float4 *p, uint64_t pol)
{
    if (POLICY == 0) return *p;
    float4 v;
    asm volatile("ld.global.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol) : "memory");
    return v;
}
template <int POLICY> __device__ __forceinline__ void stv(double2 *p, double2 v, uint64_t pol)
{
    if (POLICY == 0) { *p = v; return; }
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
template <int POLICY> __device__ __forceinline__ void stv(float4 *p, float4 v, uint64_t pol)
{
    if (POLICY == 0) { *p = v; return; }
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}

// Slab mode: the vector kernels touch only the owned x3 slices, i.e. `nseg` runs of `len` packets that
// start `off` packets into planes `stride` packets apart (layout 0: 3 complex planes; layout 1: 6 real
// planes).  len == 0: the whole vector, flat (single GPU).
struct Seg { unsigned int len, stride, off, slice; };   // slice: packets of one x3 slice of one plane
__device__ __forceinline__ size_t seg_idx(size_t k, const Seg &sg)
{
    if (sg.len == 0) return k;
    const unsigned int pl = (unsigned int)k / sg.len;
    return (size_t)pl * sg.stride + sg.off + ((unsigned int)k - pl * sg.len);
}

// Peer transport: the face push fused into the kernel that PRODUCES a vector (p in init / K2): packet k0 of the owned
// range, if it lies in the first / last owned slice, also goes (times the boundary sign) into the landing buffer of
// the rank below / above, which is laid out like a half vector of one slice.
template <typename T>
__device__ __forceinline__ void peer_store_faces(const PeerDev &pd, int kind, const Seg &sg, size_t k0, const T *v)
{
    typedef typename Pack<T>::type P;
    const int N = Pack<T>::N;
    const unsigned int pl = (unsigned int)k0 / sg.len, off = (unsigned int)k0 - pl * sg.len;
    if (off < sg.slice) {
        T w[4];
        const T s = (T)pd.sign_down;
        for (int j = 0; j < N; ++j) w[j] = s * v[j];
        reinterpret_cast<P *>(pd.land_down[kind])[(size_t)pl * sg.slice + off] = repack(w);
    }
    if (off >= sg.len - sg.slice) {
        T w[4];
        const T s = (T)pd.sign_up;
        for (int j = 0; j < N; ++j) w[j] = s * v[j];
        reinterpret_cast<P *>(pd.land_up[kind])[(size_t)pl * sg.slice + (off - (sg.len - sg.slice))] = repack(w);
    }
}

struct ShiftPtrs {
    void *x[LQCD_MAX_SHIFTS];
    void *p[LQCD_MAX_SHIFTS];
    int nshift, base;
    // rational mode (lqcd_rational_apply): y = c0 b + sum_i coef[i] x_i is accumulated instead of
    // storing the x_i; x[] is unused then
    void *y;
    double c0, coef[LQCD_MAX_SHIFTS];
};

// r = p = p_i = b, x_i = 0, rho = ||b||^2
template <typename T, int POLICY>
__global__ void __launch_bounds__(256) init_kernel(size_t npk, Seg sg, const T *__restrict__ b, T *__restrict__ r,
                                                   T *__restrict__ p, ShiftPtrs sp, SolverState *st,
                                                   double *partials, const PeerDev *pdp, int push_kind)
{
    pdl_wait();
    pdl_trigger();
    typedef typename Pack<T>::type P;
    const int N = Pack<T>::N;
    const uint64_t keep = POLICY ? l2_policy_evict_last() : 0;
    const uint64_t strm = POLICY ? l2_policy_evict_first() : 0;
    double acc = 0.0;
    T zero[4] = {0, 0, 0, 0};
    for (size_t k0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x; k0 < npk; k0 += (size_t)gridDim.x * blockDim.x) {
        const size_t k = seg_idx(k0, sg);
        P v = ldv<POLICY>(reinterpret_cast<const P *>(b) + k, keep);
        T a[4];
        unpack<T>(v, a);
        for (int j = 0; j < N; ++j) acc += (double)a[j] * (double)a[j];
        stv<POLICY>(reinterpret_cast<P *>(r) + k, v, keep);
        stv<POLICY>(reinterpret_cast<P *>(p) + k, v, keep);
        if (push_kind >= 0) peer_store_faces<T>(*pdp, push_kind, sg, k0, a);      // the faces of p = b
        if (sp.y) {
            T yy[4];
            for (int j = 0; j < N; ++j) yy[j] = (T)sp.c0 * a[j];
            stv<POLICY>(reinterpret_cast<P *>(sp.y) + k, repack(yy), strm);
        }
        for (int i = 0; i < sp.nshift; ++i) {
            if (!sp.y) stv<POLICY>(reinterpret_cast<P *>(sp.x[i]) + k, repack(zero), strm);
            if (i != sp.base) stv<POLICY>(reinterpret_cast<P *>(sp.p[i]) + k, v, strm);
        }
    }
    if (push_kind >= 0 && blockIdx.x == 0 && threadIdx.x == 0) peer_bump_halo(*pdp, push_kind);
    double total;
    if (grid_sum_last(acc, partials, &st->ticket, &total)) {
        if (st->comm) st->sum[2] = total;
        else {
            st->cur[0].rho = total;
            st->bnorm2 = total;
            if (total == 0.0) st->done = 2;
        }
    }
}

// K1: r -= alpha q ; <r,r>.  Single GPU: every CTA first adds up the <p,q> partials the Dslash left
// (`n_in` of them) and derives alpha; CTA 0 also runs the per-shift recurrence; the <r,r> partials go to
// `part_out` for K2.  Slab mode (st->comm): alpha comes from scalar_kernel, the local <r,r> goes to sum[1].
template <typename T, int POLICY>
__global__ void __launch_bounds__(256) k1_kernel(size_t npk, Seg sg, T *__restrict__ r, const T *__restrict__ q,
                                                 SolverState *st, const double *part_in, int n_in,
                                                 double *part_out, int ip, const PeerDev *pdp)
{
    pdl_wait();
    pdl_trigger();
    if (*(volatile int *)&st->done) return;
    typedef typename Pack<T>::type P;
    const int N = Pack<T>::N;
    const uint64_t keep = POLICY ? l2_policy_evict_last() : 0;
    const int comm = st->comm;
    double alpha_d;
    if (comm == 1) alpha_d = st->alpha;
    else {
        double pq;
        if (comm == 2) {     // peer transport: every CTA adds up this rank's Dslash partials (as on one GPU), CTA 0
            const double local = sum_partials(part_in, n_in);      // publishes the sum, all gather the other ranks' sums
            if (blockIdx.x == 0 && threadIdx.x == 0) peer_publish(*pdp, 0, &local, 1);
            pq = peer_gather_with_local(*pdp, 0, local);
        } else pq = sum_partials(part_in, n_in);
        alpha_d = st->cur[ip].rho / pq;
        if (blockIdx.x == 0 && threadIdx.x == 0) solver_after_pq(st, pq, ip);
    }
    const T alpha = (T)alpha_d;
    double acc = 0.0;
    for (size_t k0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x; k0 < npk; k0 += (size_t)gridDim.x * blockDim.x) {
        const size_t k = seg_idx(k0, sg);
        T a[4], c[4];
        unpack<T>(ldv<POLICY>(reinterpret_cast<const P *>(r) + k, keep), a);
        unpack<T>(ldv<POLICY>(reinterpret_cast<const P *>(q) + k, keep), c);
        for (int j = 0; j < N; ++j) {
            a[j] = fma(-alpha, c[j], a[j]);
            acc += (double)a[j] * (double)a[j];
        }
        stv<POLICY>(reinterpret_cast<P *>(r) + k, repack(a), keep);
    }
    if (comm == 1) {
        double total;
        if (grid_sum_last(acc, part_out, &st->ticket, &total)) st->sum[1] = total;
    } else {
        const double b = block_sum(acc);
        if (threadIdx.x == 0) part_out[blockIdx.x] = b;
        if (comm == 2 && blockIdx.x == 0 && threadIdx.x == 0) peer_bump_red(*pdp, 1);
    }
}

// K2: x_i += alpha_i p_i ; p_i = zeta_i r + beta_i p_i ; p = r + beta p.  The base shift has
// zeta = 1 and p_base == p, so its direction vector is not stored.
// RAT = 1 (lqcd_rational_apply): the solutions are never stored;
// y += (c_i alpha_i) p_i replaces x_i += alpha_i p_i, which removes 96 B/site/iteration of x_i
// traffic per active shift in exchange for one read-modify-write of y.
template <typename T, int POLICY, int RAT>
__global__ void __launch_bounds__(256) k2_kernel(size_t npk, Seg sg, const T *__restrict__ r, T *__restrict__ p,
                                                 ShiftPtrs sp, SolverState *st, const double *part_in, int n_in, int ip,
                                                 const PeerDev *pdp, int push_kind)
{
    pdl_wait();
    pdl_trigger();
    if (*(volatile const int *)&st->done == 2) return;
    // Single GPU: every CTA adds up K1's <r,r> partials and derives beta and the per-shift coefficients
    // from the state of iteration parity ip; CTA 0 also advances the state (into the other buffer).
    // Slab mode: the coefficients were written by scalar_kernel after the all-reduce.
    const int comm = st->comm;
    double rho_new = 0.0, beta_d;
    if (comm == 1) beta_d = st->beta;
    else {
        if (comm == 2) {     // peer transport: as in K1, with K1's partials
            const double local = sum_partials(part_in, n_in);
            if (blockIdx.x == 0 && threadIdx.x == 0) peer_publish(*pdp, 1, &local, 1);
            rho_new = peer_gather_with_local(*pdp, 1, local);
        } else rho_new = sum_partials(part_in, n_in);
        beta_d = rho_new / st->cur[ip].rho;
    }
    typedef typename Pack<T>::type P;
    const int N = Pack<T>::N;
    // r and p are re-read by the next kernels: keep.  x_i, p_i are touched once per iteration and
    // together exceed L2 for several shifts: stream them through.
    const uint64_t keep = POLICY ? l2_policy_evict_last() : 0;
    const uint64_t strm = POLICY ? l2_policy_evict_first() : 0;
    // Coefficients of the ACTIVE non-base shifts, compacted, so that the loop below is branch-free
    // and can issue the loads of K2_BATCH shifts before the first dependent FMA (the pointers may
    // alias as far as the compiler knows, so it cannot hoist loads over stores by itself).
    __shared__ T s_alpha[LQCD_MAX_SHIFTS], s_zeta[LQCD_MAX_SHIFTS], s_beta[LQCD_MAX_SHIFTS];
    __shared__ P *s_x[LQCD_MAX_SHIFTS], *s_p[LQCD_MAX_SHIFTS];
    __shared__ int s_n, s_base_active;
    __shared__ T s_base_alpha;
    if (threadIdx.x == 0) {
        int n = 0, ba = 0;
        for (int i = 0; i < sp.nshift; ++i) {
            double c_zeta, c_beta;
            int c_active;
            if (comm == 1) { c_active = st->c_active[i]; c_zeta = st->c_zeta[i]; c_beta = st->c_beta[i]; }
            else {       // same expressions as solver_after_rr
                const double zn = st->zeta_new[i], ratio = zn / st->cur[ip].zeta[i];
                c_active = st->cur[ip].active[i];
                c_zeta = zn;
                c_beta = beta_d * ratio * ratio;
            }
            if (!c_active) continue;
            const T al = RAT ? (T)(sp.coef[i] * st->c_alpha[i]) : (T)st->c_alpha[i];
            if (i == sp.base) { ba = 1; s_base_alpha = al; continue; }
            s_alpha[n] = al;
            s_zeta[n] = (T)c_zeta;
            s_beta[n] = (T)c_beta;
            s_x[n] = RAT ? (P *)0 : reinterpret_cast<P *>(sp.x[i]);
            s_p[n] = reinterpret_cast<P *>(sp.p[i]);
            ++n;
        }
        s_n = n;
        s_base_active = ba;
        // cur[ip] is not written by anyone in this kernel; the new state goes to cur[ip^1]
        if (comm != 1 && blockIdx.x == 0) solver_after_rr(st, rho_new, ip);
    }
    __syncthreads();
    const int n_act = s_n, base_active = s_base_active;
    const T beta = (T)beta_d, base_alpha = base_active ? s_base_alpha : (T)0;
    P *const xb = RAT ? reinterpret_cast<P *>(sp.y) : reinterpret_cast<P *>(sp.x[sp.base]);
    constexpr int B = 4;     // shifts whose loads are in flight together
    for (size_t k0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x; k0 < npk; k0 += (size_t)gridDim.x * blockDim.x) {
        const size_t k = seg_idx(k0, sg);
        T rr[4], pp[4], acc[4];
        unpack<T>(ldv<POLICY>(reinterpret_cast<const P *>(r) + k, keep), rr);
        unpack<T>(ldv<POLICY>(reinterpret_cast<const P *>(p) + k, keep), pp);
        // the vector the base shift updates: x_base (or y, which also collects every other shift)
        const bool touch = RAT ? true : (base_active != 0);
        if (touch) {
            unpack<T>(ldv<POLICY>(xb + k, strm), acc);
            for (int j = 0; j < N; ++j) acc[j] = fma(base_alpha, pp[j], acc[j]);
        }
        for (int a0 = 0; a0 < n_act; a0 += B) {
            P vx[B], vp[B];
#pragma unroll
            for (int u = 0; u < B; ++u)
                if (a0 + u < n_act) {
                    vp[u] = ldv<POLICY>(s_p[a0 + u] + k, strm);
                    if (!RAT) vx[u] = ldv<POLICY>(s_x[a0 + u] + k, strm);
                }
#pragma unroll
            for (int u = 0; u < B; ++u)
                if (a0 + u < n_act) {
                    T pi[4], xx[4];
                    unpack<T>(vp[u], pi);
                    if (!RAT) unpack<T>(vx[u], xx);
                    const T al = s_alpha[a0 + u], ze = s_zeta[a0 + u], be = s_beta[a0 + u];
                    for (int j = 0; j < N; ++j) {
                        if (RAT) acc[j] = fma(al, pi[j], acc[j]); else xx[j] = fma(al, pi[j], xx[j]);
                        pi[j] = fma(be, pi[j], ze * rr[j]);
                    }
                    stv<POLICY>(s_p[a0 + u] + k, repack(pi), strm);
                    if (!RAT) stv<POLICY>(s_x[a0 + u] + k, repack(xx), strm);
                }
        }
        if (touch) stv<POLICY>(xb + k, repack(acc), strm);
        for (int j = 0; j < N; ++j) pp[j] = fma(beta, pp[j], rr[j]);
        stv<POLICY>(reinterpret_cast<P *>(p) + k, repack(pp), keep);
        if (push_kind >= 0) peer_store_faces<T>(*pdp, push_kind, sg, k0, pp);     // the faces of the new p
    }
    if (push_kind >= 0 && blockIdx.x == 0 && threadIdx.x == 0) peer_bump_halo(*pdp, push_kind);
}

// Slab mode: the scalar step that the last CTA of a reduction performs on a single GPU, run after the
// caller's all-reduce of st->sum[which] (0: after <p,q>; 1: after <r,r>; 2: after <b,b>).
__global__ void scalar_kernel(SolverState *st, int which, int ip)
{
    pdl_wait();
    pdl_trigger();
    if (threadIdx.x || blockIdx.x) return;
    if (which == 2) {
        const double t = st->sum[2];
        st->cur[0].rho = t;
        st->bnorm2 = t;
        if (t == 0.0) st->done = 2;
        return;
    }
    if (*(volatile int *)&st->done) return;
    if (which == 0) solver_after_pq(st, st->sum[0], ip); else solver_after_rr(st, st->sum[1], ip);
}

// ||a - b||^2 -> *slot
template <typename T, int POLICY>
__global__ void __launch_bounds__(256) diffnorm_kernel(size_t npk, Seg sg, const T *__restrict__ a, const T *__restrict__ b,
                                                       SolverState *st, double *partials, double *slot)
{
    pdl_wait();
    pdl_trigger();
    typedef typename Pack<T>::type P;
    const int N = Pack<T>::N;
    const uint64_t keep = POLICY ? l2_policy_evict_last() : 0;
    double acc = 0.0;
    for (size_t k0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x; k0 < npk; k0 += (size_t)gridDim.x * blockDim.x) {
        const size_t k = seg_idx(k0, sg);
        T x[4], y[4];
        unpack<T>(ldv<POLICY>(reinterpret_cast<const P *>(a) + k, keep), x);
        unpack<T>(ldv<POLICY>(reinterpret_cast<const P *>(b) + k, keep), y);
        for (int j = 0; j < N; ++j) { double d = (double)x[j] - (double)y[j]; acc += d * d; }
    }
    double total;
    if (grid_sum_last(acc, partials, &st->ticket, &total)) *slot = total;
}

// ---------------------------------------------------------------------------------------------
// Host driver
// ---------------------------------------------------------------------------------------------
// Grid of a grid-stride vector kernel: ONE resident wave.  The CTAs per SM come from the occupancy
// calculator for that kernel (registers decide: k1 40 regs -> 6, k2 44 regs -> 5 CTAs of 256), capped
// by option blas_ctas_per_sm.  (Round-1 bug found with ncu: a fixed 8 CTAs/SM gave 1.33-1.6 waves,
// i.e. a second, mostly empty pass of every vector kernel.)
template <typename K>
static int blas_grid(const lqcd_ctx *ctx, K kern, size_t npk)
{
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, ctx->blas_block, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        occ = 1;
    }
    if (occ > ctx->blas_ctas_per_sm) occ = ctx->blas_ctas_per_sm;
    size_t want = (npk + ctx->blas_block - 1) / ctx->blas_block;
    size_t cap = (size_t)ctx->num_sms * occ;
    size_t g = want < cap ? want : cap;
    if (g > (size_t)ctx->max_partials) g = ctx->max_partials;
    return g < 1 ? 1 : (int)g;
}

template <typename T>
static int solve_t(lqcd_ctx *ctx, int nshift, const double *shifts, const void *b, void *const *xs,
                   const void *links, double mass, double tol, int max_iter,
                   int *iters, int *conv_iter, double *rel_resid,
                   void *y = NULL, double c0 = 0.0, const double *coef = NULL)
{
    // vector kernels: the whole half vector, or (slab mode) only the owned x3 slices of each plane
    size_t npk = (size_t)ctx->g.Vh * 6 / Pack<T>::N;
    Seg sg = {0, 0, 0, 0};
    if (ctx->x3_lo != 0 || ctx->x3_hi != ctx->g.N3) {
        const unsigned per = ctx->layout == 0 ? 2 : 1;                 // reals per site in one plane
        const unsigned nseg = ctx->layout == 0 ? 3 : 6;
        sg.len = (unsigned)((size_t)(ctx->x3_hi - ctx->x3_lo) * ctx->g.s3 * per / Pack<T>::N);
        sg.stride = (unsigned)((size_t)ctx->g.Vh * per / Pack<T>::N);
        sg.off = (unsigned)((size_t)ctx->x3_lo * ctx->g.s3 * per / Pack<T>::N);
        sg.slice = (unsigned)((size_t)ctx->g.s3 * per / Pack<T>::N);
        npk = (size_t)nseg * sg.len;
    }
    const int peer = ctx->peer_on;
    const int comm = peer ? 2 : (ctx->allreduce_fn != NULL);      // SolverState::comm
    const int par = ctx->solve_parity;                                 // parity of x, b, p, r, q
    SolverState *const dst = ctx->d_state;
    const int block = ctx->blas_block;
    const int g_init = ctx->l2_hints ? blas_grid(ctx, init_kernel<T, 1>, npk) : blas_grid(ctx, init_kernel<T, 0>, npk);
    const int g_k1 = ctx->l2_hints ? blas_grid(ctx, k1_kernel<T, 1>, npk) : blas_grid(ctx, k1_kernel<T, 0>, npk);
    const int g_k2 = y ? (ctx->l2_hints ? blas_grid(ctx, k2_kernel<T, 1, 1>, npk) : blas_grid(ctx, k2_kernel<T, 0, 1>, npk))
                       : (ctx->l2_hints ? blas_grid(ctx, k2_kernel<T, 1, 0>, npk) : blas_grid(ctx, k2_kernel<T, 0, 0>, npk));
    const int g_diff = blas_grid(ctx, diffnorm_kernel<T, 0>, npk);
    // slab hooks: ghost slices of a vector before it is a Dslash input; global sum of a local dot product
    auto halo = [&](void *v, int parity, int gate) -> int {
        if (peer) return launch_peer_push(ctx, v, parity, gate);
        if (!ctx->halo_fn) return LQCD_OK;
        if (ctx->halo_fn(ctx->comm_user, v, parity)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "halo hook failed");
        return LQCD_OK;
    };
    auto reduce_then = [&](int which, int ip) -> int {
        if (!comm) return LQCD_OK;
        if (peer) {          // <p,q> and <r,r> are gathered by the consumer kernels; <b,b> by a pair of one-CTA kernels
            if (which == 2) return launch_peer_allreduce(ctx, &dst->sum[2], 1, 1);
            // lock-step validation: the rank's sum is published before the host barrier (peer.cu); in production
            // CTA 0 of the consumer kernel does it
            return which == 0 ? launch_peer_early_publish(ctx, 0, ctx->d_partials, ctx->last_dslash_grid)
                              : launch_peer_early_publish(ctx, 1, ctx->d_partials + ctx->max_partials, g_k1);
        }
        if (ctx->allreduce_fn(ctx->comm_user, &dst->sum[which], 1)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "allreduce hook failed");
        launch_k(ctx, scalar_kernel, dim3(1), dim3(32), dst, which, ip);
        return lqcd_check_cuda(ctx, cudaGetLastError(), "scalar kernel");
    };
    cudaStream_t s = ctx->stream;
    T *tmp_o = (T *)ws_vec(ctx, 0), *q = (T *)ws_vec(ctx, 1), *r = (T *)ws_vec(ctx, 2), *p = (T *)ws_vec(ctx, 3);

    // base system = smallest shift (reading R11)
    int base = 0;
    for (int i = 1; i < nshift; ++i) if (shifts[i] < shifts[base]) base = i;
    SolverState h;
    memset(&h, 0, sizeof(h));
    h.alpha_prev = 1.0; h.beta_prev = 0.0; h.tol = tol; h.nshift = nshift;
    h.comm = comm;
    ShiftPtrs sp;
    memset(&sp, 0, sizeof(sp));
    sp.nshift = nshift; sp.base = base;
    for (int i = 0; i < nshift; ++i) {
        h.cur[0].zeta[i] = h.cur[1].zeta[i] = h.zeta_old[i] = 1.0;
        h.delta[i] = shifts[i] - shifts[base];
        h.cur[0].active[i] = h.cur[1].active[i] = 1;
        sp.x[i] = y ? NULL : xs[i];
        sp.p[i] = ws_vec(ctx, 4 + i);
        if (y) sp.coef[i] = coef[i];
    }
    sp.y = y;
    sp.c0 = c0;
    int rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(ctx->d_state, &h, sizeof(h), cudaMemcpyHostToDevice, s), "solver state upload");
    if (rc) return rc;
    const int push_kind = peer ? par : -1;     // peer transport: init and K2 push the faces of p themselves
    if (peer && (rc = peer_guard(ctx, par))) return rc;
    if (ctx->l2_hints) launch_k(ctx, init_kernel<T, 1>, dim3(g_init), dim3(block), npk, sg, (const T *)b, r, p, sp, ctx->d_state, ctx->d_partials, (const PeerDev *)ctx->d_peer, push_kind);
    else launch_k(ctx, init_kernel<T, 0>, dim3(g_init), dim3(block), npk, sg, (const T *)b, r, p, sp, ctx->d_state, ctx->d_partials, (const PeerDev *)ctx->d_peer, push_kind);
    if (peer && (rc = peer_after_producer(ctx, par, 0))) return rc;
    if ((rc = reduce_then(2, 0))) return rc;

    const double msq = mass * mass + shifts[base];
    volatile int *flag = ctx->h_flag;
    flag[0] = flag[16 / 4] = 0;
    flag[1] = flag[16 / 4 + 1] = 0;
    int enq = 0, chunk_id = 0, stop = 0;
    // one CG iteration = 4 kernels; all arguments are the same in every iteration
    // <p,q> partials (one per Dslash CTA) and <r,r> partials (one per K1 CTA) live in separate halves of
    // d_partials: K1 reads the first while it writes the second.
    double *const part_pq = ctx->d_partials, *const part_rr = ctx->d_partials + ctx->max_partials;
    auto enqueue_iteration = [&](int ip) -> int {      // ip = parity of the iteration number
        int e;
        const int m = ctx->iter_mask;   // diagnostic: which of the 4 kernels run (timing experiments only)
        // peer transport: the faces of p were pushed by its producer (init / K2), K_A pushes those of tmp_o
        if (!peer && (e = halo(p, par, 1))) return e;
        if ((m & 1) && (e = launch_dslash(ctx, 1 - par, tmp_o, p, links, NULL, 0.0, 0, 2, -1, -1, peer))) return e;
        if (peer) { if ((e = peer_after_producer(ctx, 1 - par, 1))) return e; }
        else if ((e = halo(tmp_o, 1 - par, 1))) return e;
        if ((m & 2) && (e = launch_dslash(ctx, par, q, tmp_o, links, p, msq, 1, 1))) return e;
        const int n_pq = ctx->last_dslash_grid;
        if ((e = reduce_then(0, ip))) return e;
#define K1(POL) launch_k(ctx, k1_kernel<T, POL>, dim3(g_k1), dim3(block), npk, sg, r, (const T *)q, dst, \
                         (const double *)part_pq, n_pq, part_rr, ip, (const PeerDev *)ctx->d_peer)
#define K2(POL, RAT) launch_k(ctx, k2_kernel<T, POL, RAT>, dim3(g_k2), dim3(block), npk, sg, (const T *)r, p, sp, dst, \
                              (const double *)part_rr, g_k1, ip, (const PeerDev *)ctx->d_peer, push_kind)
        if (ctx->l2_hints && !comm) {
            if (m & 4) K1(1);
            if (m & 8) { if (sp.y) K2(1, 1); else K2(1, 0); }
        } else {
            if (m & 4) K1(0);
            if ((e = reduce_then(1, ip))) return e;    // slab mode: the all-reduce of <r,r> sits between K1 and K2
            if (m & 8) { if (sp.y) K2(0, 1); else K2(0, 0); }
        }
#undef K1
#undef K2
        if (peer && (e = peer_after_producer(ctx, par, 1))) return e;
        return lqcd_check_cuda(ctx, cudaGetLastError(), "cg iteration");
    };
    // Chunk graph (option `graph`): poll_chunk iterations captured once and replayed; the key is
    // every value the captured launches depend on.
    unsigned long long key[48];
    int kn = 0;
    key[kn++] = (unsigned long long)(uintptr_t)ctx->ws; key[kn++] = (unsigned long long)(uintptr_t)links;
    key[kn++] = ((unsigned long long)ctx->x3_lo << 40) | ((unsigned long long)ctx->x3_hi << 8) | (unsigned)par;
    memcpy(&key[kn++], &msq, sizeof(double));
    key[kn++] = ((unsigned long long)nshift << 32) | (unsigned)base;
    key[kn++] = ((unsigned long long)ctx->poll_chunk << 32) | (unsigned)(g_k1 * 4096 + g_k2);
    key[kn++] = ((unsigned long long)block << 32) | (unsigned)(ctx->dslash_block * 64 + ctx->dslash_minblocks * 8 + ctx->l2_hints * 4 + ctx->pdl * 2) ^ ((unsigned long long)ctx->dslash_persist << 48);
    key[kn++] = (unsigned long long)(uintptr_t)ctx->stream ^ ((unsigned long long)ctx->iter_mask << 56);
    key[kn++] = (unsigned long long)(uintptr_t)ctx->backfield;
    key[kn++] = (unsigned long long)(uintptr_t)ctx->d_peer ^ (unsigned long long)peer;
    if (y) {
        key[kn++] = (unsigned long long)(uintptr_t)y;
        for (int i = 0; i < nshift; ++i) memcpy(&key[kn++], &coef[i], sizeof(double));
    } else {
        for (int i = 0; i < nshift; ++i) key[kn++] = (unsigned long long)(uintptr_t)xs[i];
    }
    ctx->graph_active = 0;
    // (even chunk length: the iteration parity `ip` of every captured launch is then the same in every replay)
    // (peer transport: the waits are inside the kernels, so the chunk graph stays on -- unless the lock-step
    // validation hook wants the host between the kernels)
    const bool use_graph = ctx->graph && max_iter >= ctx->poll_chunk && (comm == 0 || (peer && !ctx->phase_fn)) && !ctx->halo_fn &&
                           ctx->poll_chunk % 2 == 0;
    if (use_graph) {
        if (!ctx->chunk_exec || ctx->chunk_key_n != kn || memcmp(ctx->chunk_key, key, kn * sizeof(key[0]))) {
            if (ctx->chunk_exec) { cudaGraphExecDestroy(ctx->chunk_exec); ctx->chunk_exec = NULL; }
            const long launches0 = ctx->launches;
            cudaGraph_t g = NULL;
            int ok = cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
            if (ok) {
                ctx->launch_stream = ctx->cap_stream;
                ctx->capturing = 1;
                for (int k = 0; k < ctx->poll_chunk && ok; ++k) ok = enqueue_iteration(k & 1) == LQCD_OK;
                ctx->launch_stream = ctx->stream;
                ctx->capturing = 0;
                ok = (cudaStreamEndCapture(ctx->cap_stream, &g) == cudaSuccess) && ok && g;
            }
            if (ok) ok = cudaGraphInstantiate(&ctx->chunk_exec, g, 0) == cudaSuccess;
            if (g) cudaGraphDestroy(g);
            ctx->launches = launches0;
            if (!ok) { cudaGetLastError(); ctx->chunk_exec = NULL; ctx->graph = 0; }   // plain launches from now on
            else { memcpy(ctx->chunk_key, key, kn * sizeof(key[0])); ctx->chunk_key_n = kn; }
        }
    }
    while (!stop) {
        int n = ctx->poll_chunk;
        if (enq + n > max_iter) n = max_iter - enq;
        if (use_graph && ctx->graph && ctx->chunk_exec && n == ctx->poll_chunk) {
            if ((rc = lqcd_check_cuda(ctx, cudaGraphLaunch(ctx->chunk_exec, s), "chunk graph launch"))) return rc;
            ctx->launches += (long)__builtin_popcount(ctx->iter_mask) * n;
            ctx->graph_active = 1;
        } else {
            for (int k = 0; k < n; ++k) if ((rc = enqueue_iteration((enq + k) & 1))) return rc;
        }
        enq += n;
        int slot = chunk_id & 1;
        cudaMemcpyAsync((void *)(flag + slot * 4), &ctx->d_state->done, sizeof(int), cudaMemcpyDeviceToHost, s);
        // peer transport: a wait that gave up (peer.cuh) ends the solve at the next poll, not after max_iter iterations
        if (peer) cudaMemcpyAsync((void *)(flag + slot * 4 + 1), &((PeerBlock *)ctx->peer_mem)->timeouts, sizeof(int), cudaMemcpyDeviceToHost, s);
        cudaEventRecord(ctx->ev[slot], s);
        // look at the PREVIOUS chunk's flag, so that one chunk is always queued behind the GPU
        if (chunk_id > 0) {
            int prev = (chunk_id - 1) & 1;
            if ((rc = lqcd_check_cuda(ctx, cudaEventSynchronize(ctx->ev[prev]), "cg poll"))) return rc;
            if (flag[prev * 4] || (peer && flag[prev * 4 + 1])) stop = 1;
        }
        if (enq >= max_iter) stop = 1;
        ++chunk_id;
    }
    // (peer transport: the loop's last exchange -- K2's faces of p -- has no reader: the next K_A is gated off or was
    // never enqueued; inside the loop the kinds alternate, p / D p / p / ...)
    if (peer) ctx->peer_last_kind = -1;
    // true residuals || b - (A + sigma_i) x_i || (reading R10), with the same kernels, ungated
    for (int i = 0; i < nshift && !y; ++i) {
        if ((rc = halo(xs[i], par, 0))) return rc;
        if ((rc = launch_dslash(ctx, 1 - par, tmp_o, xs[i], links, NULL, 0.0, 0, 0))) return rc;
        if ((rc = halo(tmp_o, 1 - par, 0))) return rc;
        if ((rc = launch_dslash(ctx, par, q, tmp_o, links, xs[i], mass * mass + shifts[i], 0, 0))) return rc;
        launch_k(ctx, diffnorm_kernel<T, 0>, dim3(g_diff), dim3(block), npk, sg, (const T *)b, (const T *)q, ctx->d_state, ctx->d_partials, &ctx->d_state->resid[i]);
    }
    if (peer && !y) { if ((rc = launch_peer_allreduce(ctx, &dst->resid[0], nshift, 0))) return rc; }
    else if (comm && !y && ctx->allreduce_fn(ctx->comm_user, &dst->resid[0], nshift)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "allreduce hook failed");
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(&h, ctx->d_state, sizeof(h), cudaMemcpyDeviceToHost, s), "solver state download"))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaStreamSynchronize(s), "cg"))) return rc;

    if (iters) *iters = h.iter;
    int converged = (h.done != 0);
    for (int i = 0; i < nshift; ++i) {
        if (conv_iter) conv_iter[i] = h.cur[h.iter & 1].active[i] ? h.iter : h.conv_iter[i];
        if (rel_resid && !y) rel_resid[i] = h.bnorm2 > 0.0 ? sqrt(h.resid[i] / h.bnorm2) : 0.0;
    }
    ctx->hist_n = h.iter < LQCD_HIST ? h.iter : LQCD_HIST;
    memcpy(ctx->h_hist[0], h.hist_alpha, sizeof(h.hist_alpha));
    memcpy(ctx->h_hist[1], h.hist_beta, sizeof(h.hist_beta));
    memcpy(ctx->h_hist[2], h.hist_rnorm, sizeof(h.hist_rnorm));
    if (peer) {      // a wait for a peer gave up (dead or desynchronised rank): the results are meaningless
        const long nt = peer_timeouts(ctx);
        if (nt != 0) {      // the transport stays dead (peer.cuh): every later solve reports it again
            ctx->peer_timeouts_seen = nt;
            return lqcd_fail(ctx, LQCD_ERR_CUDA, "peer transport: %ld waits for other ranks timed out; the transport is dead until lqcd_peer_disconnect + lqcd_peer_init", nt);
        }
    }
    if (!converged) return lqcd_fail(ctx, LQCD_ERR_NOT_CONVERGED, "not converged after %d iterations", h.iter);
    return LQCD_OK;
}

// Argument hygiene shared by the solver entry points (before any launch): the vector kernels declare their
// operands __restrict__ and use 16-byte loads, so a buffer that aliases another operand, the workspace or
// the link field would corrupt the solve silently and a misaligned one would fault asynchronously.
static int check_solver_buffers(lqcd_ctx *ctx, const char *who, int n_out, void *const *outs, const void *rhs, const void *links)
{
    const uintptr_t vb = (uintptr_t)lqcd_spinor_bytes(ctx), lb = (uintptr_t)lqcd_links_bytes(ctx);
    const uintptr_t ws0 = (uintptr_t)ctx->ws, ws1 = ws0 + ctx->ws_bytes;
    const uintptr_t r0 = (uintptr_t)rhs, l0 = (uintptr_t)links;
    if ((r0 & 15) || (l0 & 15)) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: rhs / links not 16-byte aligned", who);
    if (r0 < ws1 && r0 + vb > ws0) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: rhs lies inside the workspace", who);
    if (l0 < ws1 && l0 + lb > ws0) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: links overlap the workspace", who);
    for (int i = 0; i < n_out; ++i) {
        const uintptr_t a = (uintptr_t)outs[i];
        if (!a) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: output vector %d is null", who, i);
        if (a & 15) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: output vector %d is not 16-byte aligned", who, i);
        if (a < r0 + vb && a + vb > r0) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: output vector %d aliases rhs", who, i);
        if (a < ws1 && a + vb > ws0) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: output vector %d lies inside the workspace", who, i);
        if (a < l0 + lb && a + vb > l0) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: output vector %d overlaps the link field", who, i);
        for (int j = 0; j < i; ++j) {
            const uintptr_t b = (uintptr_t)outs[j];
            if (a < b + vb && a + vb > b) return lqcd_fail(ctx, LQCD_ERR_ARG, "%s: output vectors %d and %d overlap", who, j, i);
        }
    }
    return LQCD_OK;
}

extern "C" int lqcd_cg_multishift(lqcd_ctx *ctx, int nshift, const double *shifts, const void *rhs_e,
                                  void *const *solutions_e, const void *links, double mass, double tol,
                                  int max_iter, int *iters, int *conv_iter, double *rel_resid)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return lqcd_fail(ctx, LQCD_ERR_ARG, "nshift %d not in [1,%d]", nshift, LQCD_MAX_SHIFTS);
    if (!shifts || !rhs_e || !solutions_e || !links) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_cg_multishift: null pointer");
    if (!(tol > 0.0)) return lqcd_fail(ctx, LQCD_ERR_ARG, "tol must be > 0");
    if (max_iter < 1) return lqcd_fail(ctx, LQCD_ERR_ARG, "max_iter must be >= 1");
    for (int i = 0; i < nshift; ++i) {
        if (!(shifts[i] >= 0.0)) return lqcd_fail(ctx, LQCD_ERR_ARG, "shift %d is negative or NaN", i);
        if (!solutions_e[i] || solutions_e[i] == rhs_e) return lqcd_fail(ctx, LQCD_ERR_ARG, "solution %d is null or aliases rhs", i);
    }
    if (!ctx->ws) return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "no workspace set");
    if (ctx->ws_bytes < lqcd_workspace_bytes(ctx, nshift))
        return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "workspace %zu bytes < %zu needed for %d shifts", ctx->ws_bytes, lqcd_workspace_bytes(ctx, nshift), nshift);
    if ((rc = check_solver_buffers(ctx, "lqcd_cg_multishift", nshift, solutions_e, rhs_e, links))) return rc;
    if (ctx->prec == LQCD_F64)
        return solve_t<double>(ctx, nshift, shifts, rhs_e, solutions_e, links, mass, tol, max_iter, iters, conv_iter, rel_resid);
    return solve_t<float>(ctx, nshift, shifts, rhs_e, solutions_e, links, mass, tol, max_iter, iters, conv_iter, rel_resid);
}

extern "C" int lqcd_rational_apply(lqcd_ctx *ctx, int nshift, const double *shifts, double c0, const double *coeffs,
                                   const void *rhs_e, void *y_e, const void *links, double mass, double tol,
                                   int max_iter, int *iters, int *conv_iter)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return lqcd_fail(ctx, LQCD_ERR_ARG, "nshift %d not in [1,%d]", nshift, LQCD_MAX_SHIFTS);
    if (!shifts || !coeffs || !rhs_e || !y_e || !links) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_rational_apply: null pointer");
    if (y_e == rhs_e) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_rational_apply: y aliases rhs");
    if (!(tol > 0.0)) return lqcd_fail(ctx, LQCD_ERR_ARG, "tol must be > 0");
    if (max_iter < 1) return lqcd_fail(ctx, LQCD_ERR_ARG, "max_iter must be >= 1");
    for (int i = 0; i < nshift; ++i) {
        if (!(shifts[i] >= 0.0)) return lqcd_fail(ctx, LQCD_ERR_ARG, "shift %d is negative or NaN", i);
        if (coeffs[i] != coeffs[i]) return lqcd_fail(ctx, LQCD_ERR_ARG, "coefficient %d is NaN", i);
    }
    if (c0 != c0) return lqcd_fail(ctx, LQCD_ERR_ARG, "c0 is NaN");
    if (!ctx->ws) return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "no workspace set");
    if (ctx->ws_bytes < lqcd_workspace_bytes(ctx, nshift))
        return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "workspace %zu bytes < %zu needed for %d shifts", ctx->ws_bytes, lqcd_workspace_bytes(ctx, nshift), nshift);
    { void *ys[1] = { y_e }; if ((rc = check_solver_buffers(ctx, "lqcd_rational_apply", 1, ys, rhs_e, links))) return rc; }
    if (ctx->prec == LQCD_F64)
        return solve_t<double>(ctx, nshift, shifts, rhs_e, NULL, links, mass, tol, max_iter, iters, conv_iter, NULL, y_e, c0, coeffs);
    return solve_t<float>(ctx, nshift, shifts, rhs_e, NULL, links, mass, tol, max_iter, iters, conv_iter, NULL, y_e, c0, coeffs);
}

extern "C" int lqcd_cg(lqcd_ctx *ctx, void *x_e, const void *b_e, const void *links, double mass,
                       double tol, int max_iter, int *iters, double *rel_resid)
{
    const double zero = 0.0;
    void *xs[1] = { x_e };
    if (ctx && !x_e) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_cg: null pointer");
    return lqcd_cg_multishift(ctx, 1, &zero, b_e, xs, links, mass, tol, max_iter, iters, NULL, rel_resid);
}

extern "C" int lqcd_solver_history(lqcd_ctx *ctx, int n, double *alpha, double *beta, double *rnorm)
{
    if (!ctx) return -LQCD_ERR_ARG;
    int m = n < ctx->hist_n ? n : ctx->hist_n;
    if (m < 0) m = 0;
    if (alpha) memcpy(alpha, ctx->h_hist[0], m * sizeof(double));
    if (beta) memcpy(beta, ctx->h_hist[1], m * sizeof(double));
    if (rnorm) memcpy(rnorm, ctx->h_hist[2], m * sizeof(double));
    return ctx->hist_n;
}
