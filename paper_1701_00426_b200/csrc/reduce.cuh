// reduce.cuh -- deterministic grid reduction with a fused scalar epilogue, and the scalar
// recurrences of CG / multi-shift CG (steps a6, a8 of SURVEY.md section 8(a); readings R10, R11, R13).
#pragma once
#include "common.cuh"

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the CTA (result valid in thread 0).  blockDim.x is a multiple of 32, <= 1024.
__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double s_w[32];
    __syncthreads();                       // s_w may still be in use from a previous call
    v = warp_sum(v);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) s_w[w] = v;
    __syncthreads();
    if (w == 0) {
        int nw = (blockDim.x + 31) >> 5;
        v = lane < nw ? s_w[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

// Every CTA contributes `v` (per thread).  Partials go to partials[blockIdx.x]; the CTA that
// takes the last ticket adds them in index order (fixed order => run-to-run deterministic,
// fp64 accumulation also for fp32 fields) and returns true in its thread 0 with *total set.
__device__ __forceinline__ bool grid_sum_last(double v, double *partials, unsigned int *ticket, double *total)
{
    __shared__ bool s_last;
    double b = block_sum(v);
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = b;
        __threadfence();
        unsigned int t = atomicInc(ticket, gridDim.x - 1);   // wraps back to 0 for the next use
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
    double s = 0.0;
    for (unsigned int k = threadIdx.x; k < gridDim.x; k += blockDim.x) s += __ldcg(partials + k);
    s = block_sum(s);
    if (threadIdx.x == 0) *total = s;
    return threadIdx.x == 0;
}

// ---- scalar recurrences (one thread) -----------------------------------------------------
// After q = A_b p and pq = Re<p,q>:   alpha = rho/pq;  zeta_i^new, alpha_i   (reading R11)
__device__ __forceinline__ void solver_after_pq(SolverState *st, double pq)
{
    double alpha = st->rho / pq;
    st->alpha = alpha;
    for (int i = 0; i < st->nshift; ++i) {
        double z = st->zeta[i], zo = st->zeta_old[i];
        double zn = z * zo * st->alpha_prev /
                    (alpha * st->beta_prev * (zo - z) + zo * st->alpha_prev * (1.0 + st->delta[i] * alpha));
        st->zeta_new[i] = zn;
        st->c_alpha[i] = alpha * zn / z;
    }
}

// After r -= alpha q and rho' = <r,r>:  beta, beta_i, history, convergence flags (sticky).
__device__ __forceinline__ void solver_after_rr(SolverState *st, double rho_new)
{
    double beta = rho_new / st->rho;
    st->beta = beta;
    int k = st->iter;
    if (k < LQCD_HIST) { st->hist_alpha[k] = st->alpha; st->hist_beta[k] = beta; st->hist_rnorm[k] = sqrt(rho_new); }
    double thresh = st->tol * sqrt(st->bnorm2);
    int n_active = 0;
    for (int i = 0; i < st->nshift; ++i) {
        double zn = st->zeta_new[i], z = st->zeta[i];
        double ratio = zn / z;
        st->c_zeta[i] = zn;
        st->c_beta[i] = beta * ratio * ratio;
        st->c_active[i] = st->active[i];          // what K2 of THIS iteration must update
        st->zeta_old[i] = z;
        st->zeta[i] = zn;
        if (st->active[i]) {
            if (fabs(zn) * sqrt(rho_new) > thresh) ++n_active;
            else { st->active[i] = 0; st->conv_iter[i] = k + 1; }
        }
    }
    st->alpha_prev = st->alpha;
    st->beta_prev = beta;
    st->rho = rho_new;
    st->iter = k + 1;
    if (n_active == 0) st->done = 1;               // K2 of this iteration still runs
}
