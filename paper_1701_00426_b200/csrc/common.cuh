// common.cuh -- private declarations shared by the translation units of liblqcd_b200.so.
// Nothing here is shared with oracle/ (which is plain C and has its own everything).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/lqcd.h"
#include "../../include/lqcd_diag.h"

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
    int Ls;               // link plane stride in sites (Vh + link_pad): breaks the power-of-two plane spacing
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

// ---- loads / stores with cache policy -----------------------------------------------------
// Links are read exactly once per Dslash; half-lattice vectors are re-read (8 neighbours, and by
// the next kernel of a CG iteration).  POLICY selects how that is told to the memory system:
//   POLICY 0: links ld.global.cs (streaming, evict-first), vectors ld.global.nc / plain stores
//   POLICY 1: explicit L2 cache hints (createpolicy): links L2::evict_first + L1::no_allocate,
//             vectors L2::evict_last on loads AND stores, so that the 126 MB L2 keeps the
//             25 MB vectors of a 32^4 lattice resident while 604 MB of links stream through.
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
struct L2Pol { uint64_t stream, keep; };
__device__ __forceinline__ L2Pol make_l2pol() { L2Pol p; p.stream = l2_policy_evict_first(); p.keep = l2_policy_evict_last(); return p; }

__device__ __forceinline__ double2 ld_hint_stream(const double2 *p, uint64_t pol)
{
    double2 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_hint_stream(const float2 *p, uint64_t pol)
{
    float2 v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double ld_hint_stream(const double *p, uint64_t pol)
{
    double v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float ld_hint_stream(const float *p, uint64_t pol)
{
    float v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 ld_hint_keep(const double2 *p, uint64_t pol)
{
    double2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_hint_keep(const float2 *p, uint64_t pol)
{
    float2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double ld_hint_keep(const double *p, uint64_t pol)
{
    double v;
    asm("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float ld_hint_keep(const float *p, uint64_t pol)
{
    float v;
    asm("ld.global.nc.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ void st_hint_keep(double2 *p, double2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint_keep(float2 *p, float2 v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1,%2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint_keep(double *p, double v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint_keep(float *p, float v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory");
}

// STREAM = 1: link load; 0: vector load.
template <typename T, int LAYOUT, int STREAM, int POLICY>
__device__ __forceinline__ Cx<T> ld_cx(const T *__restrict__ base, size_t plane, size_t Vh, size_t i, const L2Pol &pol)
{
    Cx<T> z;
    if (LAYOUT == 0) {
        typedef typename Vec2<T>::type V2;
        const V2 *p = reinterpret_cast<const V2 *>(base) + plane * Vh + i;
        V2 v;
        if (POLICY == 0) v = STREAM ? __ldcs(p) : __ldg(p);
        else v = STREAM ? ld_hint_stream(p, pol.stream) : ld_hint_keep(p, pol.keep);
        z.re = v.x; z.im = v.y;
    } else {
        const T *p = base + (2 * plane) * Vh + i;
        if (POLICY == 0) {
            z.re = STREAM ? __ldcs(p) : __ldg(p);
            z.im = STREAM ? __ldcs(p + Vh) : __ldg(p + Vh);
        } else {
            z.re = STREAM ? ld_hint_stream(p, pol.stream) : ld_hint_keep(p, pol.keep);
            z.im = STREAM ? ld_hint_stream(p + Vh, pol.stream) : ld_hint_keep(p + Vh, pol.keep);
        }
    }
    return z;
}
template <typename T, int LAYOUT, int POLICY>
__device__ __forceinline__ void st_cx(T *__restrict__ base, size_t plane, size_t Vh, size_t i, Cx<T> z, const L2Pol &pol)
{
    if (LAYOUT == 0) {
        typedef typename Vec2<T>::type V2;
        V2 v; v.x = z.re; v.y = z.im;
        V2 *p = reinterpret_cast<V2 *>(base) + plane * Vh + i;
        if (POLICY == 0) *p = v; else st_hint_keep(p, v, pol.keep);
    } else {
        T *p = base + (2 * plane) * Vh + i;
        if (POLICY == 0) { p[0] = z.re; p[Vh] = z.im; }
        else { st_hint_keep(p, z.re, pol.keep); st_hint_keep(p + Vh, z.im, pol.keep); }
    }
}

// ------------------------------------------------------------------------------------------
// Device-resident solver state (scalars of CG / multi-shift CG; reading R10, R11 of DESIGN.md).
// ------------------------------------------------------------------------------------------
#define LQCD_HIST 64
struct SolverState {
    // recurrence state
    // rho, zeta_i and the sticky active flags are DOUBLE-BUFFERED by iteration parity: the kernel that
    // finishes iteration k (K2) reads cur[k&1] in every CTA while its CTA 0 writes cur[(k+1)&1], so the
    // scalar step needs no grid-wide synchronisation (reduce.cuh).
    struct Recur { double rho; double zeta[LQCD_MAX_SHIFTS]; int active[LQCD_MAX_SHIFTS]; } cur[2];
    double alpha_prev, beta_prev, bnorm2, tol;
    double zeta_old[LQCD_MAX_SHIFTS], zeta_new[LQCD_MAX_SHIFTS], delta[LQCD_MAX_SHIFTS];
    // coefficients of the current iteration, written by the reduction epilogues, read by K1/K2
    double alpha, beta;
    double c_alpha[LQCD_MAX_SHIFTS], c_zeta[LQCD_MAX_SHIFTS], c_beta[LQCD_MAX_SHIFTS];
    int c_active[LQCD_MAX_SHIFTS];
    int conv_iter[LQCD_MAX_SHIFTS];
    int nshift, iter;
    int done;              // 0 running; 1 converged in this iteration (K2 still to run); 2 finished
    unsigned int ticket;   // last-block-done counter of the reductions
    int comm;              // slab mode.  1 (hooks): reductions leave LOCAL sums in sum[] (0: <p,q>, 1: <r,r>, 2: <b,b>); the
    double sum[4];         // recurrences run in scalar_kernel after the caller's all-reduce.  2 (peer transport):
                           // the producer leaves per-CTA partials; CTA 0 of the CONSUMER kernel publishes the rank's sum to
                           // every rank, every CTA of the consumer gathers the other ranks' sums (peer.cuh)
    double resid[LQCD_MAX_SHIFTS];  // ||b - (A+sigma_i) x_i||^2 recomputed at exit
    double hist_alpha[LQCD_HIST], hist_beta[LQCD_HIST], hist_rnorm[LQCD_HIST];
};

// ------------------------------------------------------------------------------------------
// Slab mode, peer-to-peer transport (peer.cuh; lqcd_peer_* in lqcd.h).  One PeerBlock per rank, in that rank's
// device memory, written by the other ranks of the node through peer / IPC mappings; the landing buffers of the
// halo faces follow it in the same allocation.
// ------------------------------------------------------------------------------------------
#define LQCD_MAX_RANKS 16
struct PeerBlock {
    unsigned int flag_halo[2][2];                 // [exchange kind = parity of the pushed vector][0: from down, 1: from up]
    unsigned int flag_red[3][LQCD_MAX_RANKS];     // [0: <p,q>, 1: <r,r>, 2: generic][sender]: the sender's counter
    unsigned int cnt_halo[2], cnt_red[3];         // LOCAL counters (only this rank writes them)
    unsigned int ticket;
    unsigned int timeouts;                        // waits of THIS rank that gave up (peer.cuh: a dead or desynchronised peer must not hang the GPU)
    unsigned int pad_[1];
    double slot[3][2][LQCD_MAX_RANKS][LQCD_MAX_SHIFTS];   // [kind][counter parity][sender][value]
};
struct PeerDev {                                  // lives in device memory (ctx->d_peer); kernels get a pointer
    int nranks, rank;
    PeerBlock *self;
    PeerBlock *peer[LQCD_MAX_RANKS];              // peer[rank] == self
    void *land_self[2][2];                        // my landing buffers [kind][0: from down, 1: from up]
    void *land_up[2], *land_down[2];              // [kind]: up neighbour's "from down" buffer, down neighbour's "from up" buffer
    PeerBlock *up, *down;
    double sign_up, sign_down;                    // boundary sign applied by the SENDER to the face sent up / down
    long long wait_cycles;                        // longest wait for a peer, in SM clock cycles (option peer_wait_ms)
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
    int link_pad;          // extra sites between link planes
    int l2_persist;        // 1: persisting-L2 access-policy window over the CG vectors
    long l2_window_bytes, l2_max_persist;
    int l2_saved;          // apply_l2_window saved the device limit / stream window it found:
    size_t l2_prev_limit;
    cudaStreamAttrValue l2_prev_attr;
    int l2_hints;          // 0: ld.cs / plain, 1: explicit L2 evict_first / evict_last hints
    int dslash_block;      // threads per CTA of the Dslash kernel
    int dslash_minblocks;  // launch-bounds variant (occupancy target)
    int blas_block, blas_ctas_per_sm;
    int poll_chunk;        // CG iterations enqueued between convergence polls
    int pdl;               // 1: programmatic dependent launch (kernel N+1 is scheduled while N drains)
    int capturing;         // (internal) launches are being captured into the chunk graph: plain edges there --
                           // inside a graph PDL gains nothing and costs 4 us per iteration at 16^4 (experiments_r1b.md section 8)
    int graph;             // 1: the solver replays one CUDA graph per chunk of poll_chunk iterations
    int dslash_persist;    // 0: one 128-site tile per CTA; k > 0: num_sms*k CTAs loop over the tiles
    // slab mode (multi-GPU): the context describes the rank's x3 slab plus one
    // ghost slice on each side; only the slices [x3_lo, x3_hi) are owned (default: all of them)
    int x3_lo, x3_hi;
    int solve_parity;      // local parity of the sites the solvers act on (default LQCD_EVEN)
    // peer-to-peer transport (lqcd_peer_init / lqcd_peer_connect): library-owned block + landing buffers
    int peer_on;                     // 1 after lqcd_peer_connect: solvers, lqcd_dslash and lqcd_mdagm use it
    int peer_nranks, peer_rank;
    int peer_wait_ms;                // longest wait for a peer (default 3000 ms); takes effect at lqcd_peer_connect
    long peer_timeouts_seen;         // value of the block's timeout counter the host has already reported
    int peer_last_kind;              // kind of the most recent halo exchange whose reader may still run (-1: none); peer_guard
    double peer_sign_up, peer_sign_down;   // boundary sign applied by the SENDER to the face sent up / down
    void *peer_mem; size_t peer_mem_bytes; // cudaMalloc: PeerBlock + 4 landing buffers
    PeerDev h_peer, *d_peer;
    void *peer_opened[LQCD_MAX_RANKS];     // IPC mappings to close (NULL: not ours)
    lqcd_phase_fn phase_fn; void *phase_user;   // validation hook: called after every launch that publishes to peers
    lqcd_halo_fn halo_fn;            // fills the ghost slices of a half vector (NULL: nothing to do)
    lqcd_allreduce_fn allreduce_fn;  // sums device doubles over the ranks (NULL: single rank)
    void *comm_user;
    int backfield_format;  // 0: theta stored (one real per link, sincos in-kernel); 1: (cos theta, sin theta) stored
    int backfield_locked;  // a backfield was packed: the format can no longer change
    const void *backfield; // native U(1) phase field applied by every Dslash of this context (NULL: none; lqcd_set_backfield)
    int force_stage;       // 1: force_kernel stages the site's own vectors in shared memory when they fit
    int force_block;       // right-hand sides per launch of the block Dslash that computes the y_i (0: one Dslash per shift; 4; 8)
    int staples_x2block;   // x2 block size of the staples' CTA order (0: plain idxh order)
    int staples_variant;   // 0: one product chain per path; 1: shared sub-products per (mu, nu); 2: two passes through
                           // stored 3-link staples (needs lqcd_staples_workspace_bytes of workspace, else 1 runs)
    int staples_minblocks; // launch-bounds variant (2, 3, 4 CTAs of 128 per SM) of the two-pass algorithm's second kernel; 0: default
    int staples_ran;       // read-only: the variant the last lqcd_gauge_staples call used
    int iter_mask;         // diagnostic: bit k set = kernel k of the CG iteration is launched (default 15)
    int graph_active;      // read-only: the last solve ran from a graph
    cudaStream_t cap_stream;      // private stream used only for graph capture
    cudaStream_t launch_stream;   // where launch_k enqueues: ctx->stream, or cap_stream while capturing
    cudaGraphExec_t chunk_exec;   // cached chunk graph and the key it was built for
    unsigned long long chunk_key[48];
    int chunk_key_n;
    int num_sms;
    void *ws; size_t ws_bytes;
    SolverState *d_state;  // device
    double *d_partials;    // device, reduction partials
    int max_partials;
    int *h_flag;           // pinned host words (two poll slots)
    cudaEvent_t ev[2];
    void *stage; size_t stage_bytes;   // device staging of the *_host entry points (grow-only)
    // copy pipeline of lqcd_dslash_host_vectors_batch (created on first use): uploads and downloads run on
    // their own streams so that the D2H of application n overlaps the H2D of application n+1
    cudaStream_t h2d_stream, d2h_stream;
    cudaEvent_t pipe_ev[3][2];         // [0: upload done, 1: compute done, 2: download done][slot]
    int hist_n;
    double h_hist[3][LQCD_HIST];
    int last_dslash_grid;  // CTAs of the most recent Dslash launch (= number of <p,q> partials)
    long launches;         // kernels launched through this context (bench.py's gpu_launches)
    char err[256];
};

// ------------------------------------------------------------------------------------------
// Programmatic dependent launch (sm_90+).  Every kernel of the library starts with pdl_wait()
// -- which returns once the preceding kernel in the stream has completed and its writes are
// visible; a no-op without the launch attribute -- and calls pdl_trigger() right after, so that
// the CTAs of the NEXT kernel become resident while the last wave of this one drains and are
// parked in their own pdl_wait().  Nothing is read or written before pdl_wait(): the dependency
// semantics are exactly those of plain stream order; only launch latency and ramp-up overlap.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static inline cudaError_t launch_k_smem(lqcd_ctx *ctx, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem,
                                        Args... args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = ctx->launch_stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = (ctx->pdl && !ctx->capturing) ? 1 : 0;
    ctx->launches++;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_k(lqcd_ctx *ctx, void (*kern)(KArgs...), dim3 grid, dim3 block, Args... args)
{
    return launch_k_smem(ctx, kern, grid, block, 0, args...);
}

int lqcd_fail(lqcd_ctx *ctx, int code, const char *fmt, ...);
int lqcd_check_cuda(lqcd_ctx *ctx, cudaError_t e, const char *what);
size_t elem_size(const lqcd_ctx *ctx);

// launchers implemented in the .cu files (all enqueue on ctx->stream)
int launch_pack_links(lqcd_ctx *ctx, void *native, const void *canonical);
int launch_pack_spinor(lqcd_ctx *ctx, int parity, void *native, const void *canonical);
int launch_pack_backfield(lqcd_ctx *ctx, void *native, const void *canonical);
int launch_unpack_spinor(lqcd_ctx *ctx, int parity, void *canonical, const void *native);
// out = D in; if xpay_in != NULL: out = coef*xpay_in - D in and partial Re<xpay_in,out> is reduced
// into the solver state (dot_mode 1: CG "pq" epilogue; 0: none).  `gate`: obey state->done.
// push_out (peer transport only): the kernel also stores the two boundary slices of `out` into the neighbours'
// landing buffers (the face push fused into the producer)
int launch_dslash(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                  const void *xpay_in, double coef, int dot_mode, int gate, int x3_lo = -1, int x3_hi = -1, int push_out = 0);
// block Dslash (dslash_multi.cu): outs[r] = D ins[r], r < n, each link loaded once per block of `blk` (4 or 8) vectors
int launch_dslash_multi(lqcd_ctx *ctx, int parity, int n, void *const *outs, const void *const *ins, const void *links, int blk);
int peer_after_producer(lqcd_ctx *ctx, int kind, int gate);
long peer_timeouts(lqcd_ctx *ctx);           // waits that gave up (blocking read of the rank's block)
int peer_guard(lqcd_ctx *ctx, int kind);     // barrier before two exchanges of the same kind in a row (peer.cu)    // lock-step validation: signal kernel + host hook
int launch_halo(lqcd_ctx *ctx, int pack, void *buf, void *spinor, int x3, double sign);
// peer transport (peer.cu): push both faces of `spinor` (a vector of local parity `parity`) to the neighbours
int launch_peer_push(lqcd_ctx *ctx, const void *spinor, int parity, int gate);
int launch_peer_pull(lqcd_ctx *ctx, void *spinor, int parity);   // the faces just exchanged -> the vector's own ghost slices
int peer_phase(lqcd_ctx *ctx, int what);     // lock-step validation hook (no-op unless set)
int launch_peer_allreduce(lqcd_ctx *ctx, double *vals, int nv, int which);
int launch_peer_early_publish(lqcd_ctx *ctx, int kind, const double *partials, int n);   // lock-step validation only
void lqcd_peer_destroy(lqcd_ctx *ctx);
int launch_halo2(lqcd_ctx *ctx, int pack, void *buf0, void *buf1, void *spinor, int x3_0, int x3_1, double sign0, double sign1);
