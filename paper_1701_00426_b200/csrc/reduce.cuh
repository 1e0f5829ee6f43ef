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

// Sum of `n` per-CTA partials written by the PREVIOUS kernel, computed by every CTA for itself in the
// same fixed order (so every CTA gets the bit-identical total, run-to-run deterministic).  This replaces
// fence + ticket + last-CTA sum in the producer: the producer only stores its partial, and the serial
// tail of the reduction disappears (profiles/experiments_r1b.md section 3).  All threads get the result.
__device__ __forceinline__ double sum_partials(const double *partials, int n)
{
    __shared__ double s_total;
    double s = 0.0;
    for (int k = threadIdx.x; k < n; k += blockDim.x) s += partials[k];
    s = block_sum(s);
    if (threadIdx.x == 0) s_total = s;
    __syncthreads();
    return s_total;
}

// ---- scalar recurrences (one thread) -------------------------------------------------------
// ip = parity of the iteration number: the buffer of SolverState::cur that holds the current state.
// After q = A_b p and pq = Re<p,q>:   alpha = rho/pq;  zeta_i^new, alpha_i   (reading R11)
__device__ __forceinline__ void solver_after_pq(SolverState *st, double pq, int ip)
{
    const SolverState::Recur &c = st->cur[ip];
    double alpha = c.rho / pq;
    st->alpha = alpha;
    for (int i = 0; i < st->nshift; ++i) {
        double z = c.zeta[i], zo = st->zeta_old[i];
        double zn = z * zo * st->alpha_prev /
                    (alpha * st->beta_prev * (zo - z) + zo * st->alpha_prev * (1.0 + st->delta[i] * alpha));
        st->zeta_new[i] = zn;
        st->c_alpha[i] = alpha * zn / z;
    }
}

// After r -= alpha q and rho' = <r,r>:  beta, beta_i, history, convergence flags (sticky).
// Reads cur[ip], writes cur[ip^1].
__device__ __forceinline__ void solver_after_rr(SolverState *st, double rho_new, int ip)
{
    const SolverState::Recur &c = st->cur[ip];
    SolverState::Recur &nx = st->cur[ip ^ 1];
    double beta = rho_new / c.rho;
    st->beta = beta;
    int k = st->iter;
    if (k < LQCD_HIST) { st->hist_alpha[k] = st->alpha; st->hist_beta[k] = beta; st->hist_rnorm[k] = sqrt(rho_new); }
    double thresh = st->tol * sqrt(st->bnorm2);
    int n_active = 0;
    for (int i = 0; i < st->nshift; ++i) {
        double zn = st->zeta_new[i], z = c.zeta[i];
        double ratio = zn / z;
        int act = c.active[i];
        st->c_zeta[i] = zn;
        st->c_beta[i] = beta * ratio * ratio;
        st->c_active[i] = act;                    // what K2 of THIS iteration must update
        st->zeta_old[i] = z;
        nx.zeta[i] = zn;
        if (act) {
            if (fabs(zn) * sqrt(rho_new) > thresh) ++n_active;
            else { act = 0; st->conv_iter[i] = k + 1; }
        }
        nx.active[i] = act;
    }
    st->alpha_prev = st->alpha;
    st->beta_prev = beta;
    nx.rho = rho_new;
    st->iter = k + 1;
    if (n_active == 0) st->done = 1;               // K2 of this iteration still runs
}
