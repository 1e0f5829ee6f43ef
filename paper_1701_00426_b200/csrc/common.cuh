// common.cuh -- private declarations shared by the translation units of liblqcd_b200.so.
// Nothing here is shared with oracle/ (which is plain C and has its own everything).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/lqcd.h"

// ------------------------------------------------------------------------------------------
// Lattice geometry handed to kernels by value.
// Even/odd site index of PAPER.md:259-261 (Eq. 9): idxh = (x0 + N0*(x1 + N1*(x2 + N2*x3)))/2,
// i.e. idxh = hx0 + Nh0*(x1 + N1*(x2 + N2*x3)) with hx0 = x0/2, Nh0 = N0/2.
// ------------------------------------------------------------------------------------------
struct FastDiv {          // n / d for 0 <= n < 2^31 by multiply-high (d >= 1)
    uint32_t mul, shift, d;
};
static inline FastDiv make_fastdiv(uint32_t d)
{
    FastDiv f;
    f.d = d;
    if (d == 1) { f.mul = 0; f.shift = 0; return f; }
    uint32_t l = 0;
    while ((1u << l) < d) ++l;                 // l = ceil(log2 d)
    uint64_t m = ((uint64_t(1) << (32 + l - 1)) + d - 1) / d;  // ceil(2^(32+l-1)/d), fits 32 bits for n < 2^31
    f.mul = (uint32_t)m;
    f.shift = l - 1;
    return f;
}
__device__ __forceinline__ uint32_t fd_div(uint32_t n, const FastDiv &f)
{
    return f.d == 1 ? n : (__umulhi(n, f.mul) >> f.shift);
}

struct Geom {
    int N0, N1, N2, N3;   // extents (all even)
    int Nh0;              // N0/2
    int Vh;               // sites per parity
    int s1, s2, s3;       // idxh strides of x1, x2, x3: Nh0, Nh0*N1, Nh0*N1*N2
    int ap;               // antiperiodic in x3
    FastDiv dNh0, dN1, dN2;
};

// ------------------------------------------------------------------------------------------
// Native layout (private).  A "plane" is one complex component for all Vh sites of one parity.
//   layout 0 (interleaved): plane p, site i -> reals [ (p*Vh + i)*2 + {0:re,1:im} ]
//   layout 1 (split)      : plane p, site i -> reals [ (2p + {0,1})*Vh + i ]
// half spinor : 3 planes (colour c)
// links       : plane ((par*4 + mu)*R + row)*3 + col, R = 3 (18-real) or 2 (12-real);
//               U_mu(x) is stored at x's own parity and idxh.
// ------------------------------------------------------------------------------------------
template <typename T> struct Vec2;
template <> struct Vec2<double> { typedef double2 type; };
template <> struct Vec2<float> { typedef float2 type; };

template <typename T> struct Cx { T re, im; };

template <typename T> __device__ __forceinline__ Cx<T> cx(T re, T im) { Cx<T> z; z.re = re; z.im = im; return z; }

// ---- loads with cache policy -------------------------------------------------------------
// STREAM = 1: links, read exactly once per Dslash -> ld.global.cs (evict-first in L1/L2), so the
// 126 MB L2 keeps the input spinor, which every output site's 8 neighbours re-read.
template <typename T, int LAYOUT, int STREAM>
__device__ __forceinline__ Cx<T> ld_cx(const T *__restrict__ base, size_t plane, size_t Vh, size_t i)
{
    Cx<T> z;
    if (LAYOUT == 0) {
        typedef typename Vec2<T>::type V2;
        const V2 *p = reinterpret_cast<const V2 *>(base) + plane * Vh + i;
        V2 v = STREAM ? __ldcs(p) : __ldg(p);
        z.re = v.x; z.im = v.y;
    } else {
        const T *p = base + (2 * plane) * Vh + i;
        z.re = STREAM ? __ldcs(p) : __ldg(p);
        z.im = STREAM ? __ldcs(p + Vh) : __ldg(p + Vh);
    }
    return z;
}
template <typename T, int LAYOUT>
__device__ __forceinline__ void st_cx(T *__restrict__ base, size_t plane, size_t Vh, size_t i, Cx<T> z)
{
    if (LAYOUT == 0) {
        typedef typename Vec2<T>::type V2;
        V2 v; v.x = z.re; v.y = z.im;
        reinterpret_cast<V2 *>(base)[plane * Vh + i] = v;
    } else {
        base[(2 * plane) * Vh + i] = z.re;
        base[(2 * plane + 1) * Vh + i] = z.im;
    }
}

// ------------------------------------------------------------------------------------------
// Device-resident solver state (scalars of CG / multi-shift CG; reading R10, R11 of DESIGN.md).
// ------------------------------------------------------------------------------------------
#define LQCD_HIST 64
struct SolverState {
    // recurrence state
    double rho, alpha_prev, beta_prev, bnorm2, tol;
    double zeta[LQCD_MAX_SHIFTS], zeta_old[LQCD_MAX_SHIFTS], zeta_new[LQCD_MAX_SHIFTS], delta[LQCD_MAX_SHIFTS];
    // coefficients of the current iteration, written by the reduction epilogues, read by K1/K2
    double alpha, beta;
    double c_alpha[LQCD_MAX_SHIFTS], c_zeta[LQCD_MAX_SHIFTS], c_beta[LQCD_MAX_SHIFTS];
    int c_active[LQCD_MAX_SHIFTS];
    int active[LQCD_MAX_SHIFTS], conv_iter[LQCD_MAX_SHIFTS];
    int nshift, iter;
    int done;              // 0 running; 1 converged in this iteration (K2 still to run); 2 finished
    unsigned int ticket;   // last-block-done counter of the reductions
    double resid[LQCD_MAX_SHIFTS];  // ||b - (A+sigma_i) x_i||^2 recomputed at exit
    double hist_alpha[LQCD_HIST], hist_beta[LQCD_HIST], hist_rnorm[LQCD_HIST];
};

// ------------------------------------------------------------------------------------------
// Context
// ------------------------------------------------------------------------------------------
struct lqcd_ctx {
    Geom g;
    int prec, recon, device;
    cudaStream_t stream;
    int layout;            // 0 interleaved complex, 1 split re/im
    int layout_locked;
    int dslash_block;      // threads per CTA of the Dslash kernel
    int dslash_minblocks;  // launch-bounds variant (occupancy target)
    int blas_block, blas_ctas_per_sm;
    int poll_chunk;        // CG iterations enqueued between convergence polls
    int num_sms;
    void *ws; size_t ws_bytes;
    SolverState *d_state;  // device
    double *d_partials;    // device, reduction partials
    int max_partials;
    int *h_flag;           // pinned host words (two poll slots)
    cudaEvent_t ev[2];
    void *stage; size_t stage_bytes;   // device staging of the *_host entry points (grow-only)
    int hist_n;
    double h_hist[3][LQCD_HIST];
    long launches;         // kernels launched through this context (bench.py's gpu_launches)
    char err[256];
};

int lqcd_fail(lqcd_ctx *ctx, int code, const char *fmt, ...);
int lqcd_check_cuda(lqcd_ctx *ctx, cudaError_t e, const char *what);
size_t elem_size(const lqcd_ctx *ctx);

// launchers implemented in the .cu files (all enqueue on ctx->stream)
int launch_pack_links(lqcd_ctx *ctx, void *native, const void *canonical);
int launch_pack_spinor(lqcd_ctx *ctx, int parity, void *native, const void *canonical);
int launch_unpack_spinor(lqcd_ctx *ctx, int parity, void *canonical, const void *native);
// out = D in; if xpay_in != NULL: out = coef*xpay_in - D in and partial Re<xpay_in,out> is reduced
// into the solver state (dot_mode 1: CG "pq" epilogue; 0: none).  `gate`: obey state->done.
int launch_dslash(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                  const void *xpay_in, double coef, int dot_mode, int gate);
