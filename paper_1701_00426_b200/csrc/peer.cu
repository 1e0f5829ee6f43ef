// peer.cu -- slab mode over peer-to-peer memory inside one node (the paper
// leaves the multi-device version as future work): set-up of the per-rank PeerBlock, CUDA IPC
// plumbing, the face-push kernel and the two generic publish / gather kernels.  Protocol: peer.cuh.
#include <stdlib.h>

#include "peer.cuh"
#include "reduce.cuh"
#include "su3.cuh"

static size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }
static size_t land_bytes(const lqcd_ctx *ctx) { return align256(lqcd_halo_bytes(ctx)); }
static size_t peer_block_bytes(const lqcd_ctx *ctx) { return align256(sizeof(PeerBlock)) + 4 * land_bytes(ctx); }
static void *land_ptr(const lqcd_ctx *ctx, void *block, int kind, int dir)
{
    return (char *)block + align256(sizeof(PeerBlock)) + (size_t)(kind * 2 + dir) * land_bytes(ctx);
}

extern "C" size_t lqcd_peer_block_bytes(const lqcd_ctx *ctx) { return ctx ? peer_block_bytes(ctx) : 0; }

static void peer_release(lqcd_ctx *ctx)
{
    for (int r = 0; r < LQCD_MAX_RANKS; ++r)
        if (ctx->peer_opened[r]) { cudaIpcCloseMemHandle(ctx->peer_opened[r]); ctx->peer_opened[r] = NULL; }
    if (ctx->peer_mem) cudaFree(ctx->peer_mem);
    if (ctx->d_peer) cudaFree(ctx->d_peer);
    ctx->peer_mem = NULL; ctx->d_peer = NULL; ctx->peer_on = 0; ctx->peer_nranks = 0;
}
void lqcd_peer_destroy(lqcd_ctx *ctx) { peer_release(ctx); }

extern "C" int lqcd_peer_init(lqcd_ctx *ctx, int nranks, int rank, int x3_lo, int x3_hi, int solve_parity,
                              double sign_up, double sign_down, void **block)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nranks < 1 || nranks > LQCD_MAX_RANKS || rank < 0 || rank >= nranks)
        return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_init: rank %d of %d (at most %d ranks)", rank, nranks, LQCD_MAX_RANKS);
    if (solve_parity != 0 && solve_parity != 1) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_init: solve_parity %d", solve_parity);
    if (!(1 <= x3_lo && x3_lo < x3_hi && x3_hi <= ctx->g.N3 - 1))
        return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_init: owned slices [%d,%d) need a ghost slice on each side of [0,%d)", x3_lo, x3_hi, ctx->g.N3);
    if (ctx->halo_fn) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_init: the context already uses communication hooks (lqcd_set_slab)");
    peer_release(ctx);
    cudaError_t e;
    ctx->peer_mem_bytes = peer_block_bytes(ctx);
    if ((e = cudaMalloc(&ctx->peer_mem, ctx->peer_mem_bytes)) != cudaSuccess ||
        (e = cudaMalloc(&ctx->d_peer, sizeof(PeerDev))) != cudaSuccess ||
        (e = cudaMemset(ctx->peer_mem, 0, ctx->peer_mem_bytes)) != cudaSuccess ||
        (e = cudaDeviceSynchronize()) != cudaSuccess) {
        peer_release(ctx);
        return lqcd_check_cuda(ctx, e, "lqcd_peer_init");
    }
    ctx->peer_nranks = nranks; ctx->peer_rank = rank;
    ctx->peer_last_kind = -1;
    ctx->peer_timeouts_seen = 0;
    ctx->peer_sign_up = sign_up; ctx->peer_sign_down = sign_down;
    ctx->x3_lo = x3_lo; ctx->x3_hi = x3_hi; ctx->solve_parity = solve_parity;
    if (ctx->chunk_exec) { cudaGraphExecDestroy(ctx->chunk_exec); ctx->chunk_exec = NULL; }
    if (block) *block = ctx->peer_mem;
    return LQCD_OK;
}

extern "C" int lqcd_peer_connect(lqcd_ctx *ctx, void *const *blocks)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!ctx->peer_mem) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_connect: call lqcd_peer_init first");
    if (!blocks) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_connect: null pointer");
    const int P = ctx->peer_nranks, me = ctx->peer_rank;
    PeerDev &h = ctx->h_peer;
    memset(&h, 0, sizeof(h));
    h.nranks = P; h.rank = me;
    h.self = (PeerBlock *)ctx->peer_mem;
    for (int r = 0; r < P; ++r) {
        void *b = r == me ? ctx->peer_mem : blocks[r];
        if (!b) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_connect: block of rank %d is null", r);
        h.peer[r] = (PeerBlock *)b;
    }
    const int up = (me + 1) % P, down = (me + P - 1) % P;
    h.up = h.peer[up]; h.down = h.peer[down];
    h.sign_up = ctx->peer_sign_up; h.sign_down = ctx->peer_sign_down;
    {
        int khz = 0;
        cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, ctx->device);
        h.wait_cycles = (long long)(ctx->peer_wait_ms > 0 ? ctx->peer_wait_ms : 3000) * (long long)(khz > 0 ? khz : 1900000);
    }
    for (int k = 0; k < 2; ++k) {
        for (int d = 0; d < 2; ++d) h.land_self[k][d] = land_ptr(ctx, ctx->peer_mem, k, d);
        h.land_up[k] = land_ptr(ctx, h.up, k, 0);       // my top slice is what the rank above receives "from down"
        h.land_down[k] = land_ptr(ctx, h.down, k, 1);
    }
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpy(ctx->d_peer, &h, sizeof(h), cudaMemcpyHostToDevice), "lqcd_peer_connect"))) return rc;
    ctx->peer_on = 1;
    if (ctx->chunk_exec) { cudaGraphExecDestroy(ctx->chunk_exec); ctx->chunk_exec = NULL; }
    return LQCD_OK;
}

extern "C" int lqcd_peer_disconnect(lqcd_ctx *ctx)
{
    if (!ctx) return LQCD_ERR_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    peer_release(ctx);
    ctx->x3_lo = 0; ctx->x3_hi = ctx->g.N3; ctx->solve_parity = LQCD_EVEN;
    if (ctx->chunk_exec) { cudaGraphExecDestroy(ctx->chunk_exec); ctx->chunk_exec = NULL; }
    return LQCD_OK;
}

// ---- CUDA IPC plumbing for one process per GPU -------------------------------------------------------------------
extern "C" int lqcd_peer_export(lqcd_ctx *ctx, void *handle64)
{
    if (!ctx || !handle64) return LQCD_ERR_ARG;
    if (!ctx->peer_mem) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_export: call lqcd_peer_init first");
    cudaSetDevice(ctx->device);
    cudaIpcMemHandle_t h;
    static_assert(sizeof(h) == 64, "cudaIpcMemHandle_t is 64 bytes");
    int rc = lqcd_check_cuda(ctx, cudaIpcGetMemHandle(&h, ctx->peer_mem), "cudaIpcGetMemHandle");
    if (rc) return rc;
    memcpy(handle64, &h, 64);
    return LQCD_OK;
}

extern "C" int lqcd_peer_import(lqcd_ctx *ctx, int rank, const void *handle64, void **block)
{
    if (!ctx || !handle64 || !block) return LQCD_ERR_ARG;
    if (rank < 0 || rank >= ctx->peer_nranks || rank == ctx->peer_rank) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_import: rank %d", rank);
    cudaSetDevice(ctx->device);
    cudaIpcMemHandle_t h;
    memcpy(&h, handle64, 64);
    void *p = NULL;
    int rc = lqcd_check_cuda(ctx, cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess), "cudaIpcOpenMemHandle");
    if (rc) return rc;
    if (ctx->peer_opened[rank]) cudaIpcCloseMemHandle(ctx->peer_opened[rank]);
    ctx->peer_opened[rank] = p;
    *block = p;
    return LQCD_OK;
}

extern "C" int lqcd_set_phase_hook(lqcd_ctx *ctx, lqcd_phase_fn fn, void *user)
{
    if (!ctx) return LQCD_ERR_ARG;
    ctx->phase_fn = fn; ctx->phase_user = user;
    if (ctx->chunk_exec) { cudaGraphExecDestroy(ctx->chunk_exec); ctx->chunk_exec = NULL; }
    return LQCD_OK;
}

// number of waits of this rank that gave up since lqcd_peer_init (blocking: finishes the stream first); < 0 on error
long peer_timeouts(lqcd_ctx *ctx)
{
    if (!ctx->peer_mem) return 0;
    unsigned int n = 0;
    if (cudaStreamSynchronize(ctx->stream) != cudaSuccess ||
        cudaMemcpy(&n, &((PeerBlock *)ctx->peer_mem)->timeouts, sizeof(n), cudaMemcpyDeviceToHost) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    return (long)n;
}

int peer_phase(lqcd_ctx *ctx, int what)
{
    if (!ctx->phase_fn) return LQCD_OK;
    if (ctx->phase_fn(ctx->phase_user, what)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "phase hook failed");
    return LQCD_OK;
}

// ---- face push ---------------------------------------------------------------------------------------------------
// blockIdx.y = 0: my top owned slice (x3_hi - 1), times sign_up, -> the up neighbour's "from down" landing buffer;
// blockIdx.y = 1: my bottom owned slice (x3_lo), times sign_down, -> the down neighbour's "from up" buffer.
// One thread counts the exchange; the flags are raised by the Dslash that follows (kernel boundary).
template <typename T, int LAYOUT>
__global__ void __launch_bounds__(128) peer_push_kernel(const Geom g, const PeerDev *__restrict__ pdp, const int kind,
                                                        const T *__restrict__ spinor, const int x3_lo, const int x3_hi,
                                                        const T sign_up, const T sign_down, const SolverState *__restrict__ st,
                                                        const int gate)
{
    pdl_wait();
    pdl_trigger();
    if (gate && *(volatile const int *)&st->done) return;     // a converged solve: every rank skips the same exchanges
    const PeerDev &pd = *pdp;
    const int up = blockIdx.y == 0;
    T *__restrict__ buf = reinterpret_cast<T *>(up ? pd.land_up[kind] : pd.land_down[kind]);
    const int x3 = up ? x3_hi - 1 : x3_lo;
    const T sign = up ? sign_up : sign_down;
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f < g.s3) {
        const size_t i = (size_t)x3 * g.s3 + f;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const Cx<T> z = ld_cx<T, LAYOUT, 0, 0>(spinor, (size_t)c, (size_t)g.Vh, i, L2Pol());
            st_cx<T, LAYOUT, 0>(buf, (size_t)c, (size_t)g.s3, (size_t)f, cx<T>(sign * z.re, sign * z.im), L2Pol());
        }
    }
    // no fence, no ticket: the Dslash that follows in the stream raises the flags (peer.cuh)
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) peer_bump_halo(pd, kind);
}

// Lock-step validation only (lqcd_set_phase_hook): with every rank on ONE GPU no kernel may wait for another rank's
// kernel, so what CTA 0 of the consumer does in production -- raise the halo flags, publish the rank's partial sum --
// is done by these one-CTA kernels BEFORE the host barrier; the consumer then repeats the same stores (same
// values, same counter) and finds every flag it waits for already raised.
__global__ void peer_signal_kernel(const PeerDev *pdp, int kind, const SolverState *st, int gate)
{
    pdl_wait();
    pdl_trigger();
    if (gate && *(volatile const int *)&st->done) return;
    if (threadIdx.x == 0) peer_signal_halo(*pdp, kind);
}
__global__ void peer_early_publish_kernel(const PeerDev *pdp, int kind, const double *partials, int n, const SolverState *st)
{
    pdl_wait();
    pdl_trigger();
    if (*(volatile const int *)&st->done) return;
    const double local = sum_partials(partials, n);
    if (threadIdx.x == 0) peer_publish(*pdp, kind, &local, 1);
}
int launch_peer_early_publish(lqcd_ctx *ctx, int kind, const double *partials, int n)
{
    if (!ctx->phase_fn) return LQCD_OK;
    launch_k(ctx, peer_early_publish_kernel, dim3(1), dim3(256), (const PeerDev *)ctx->d_peer, kind, partials, n, (const SolverState *)ctx->d_state);
    int rc = lqcd_check_cuda(ctx, cudaGetLastError(), "peer early publish");
    return rc ? rc : peer_phase(ctx, 2);
}

int peer_after_producer(lqcd_ctx *ctx, int kind, int gate)
{
    if (!ctx->phase_fn) return LQCD_OK;
    launch_k(ctx, peer_signal_kernel, dim3(1), dim3(32), (const PeerDev *)ctx->d_peer, kind, (const SolverState *)ctx->d_state, gate);
    int rc = lqcd_check_cuda(ctx, cudaGetLastError(), "peer signal");
    return rc ? rc : peer_phase(ctx, 0);
}

// A landing buffer may be rewritten only after the neighbour's Dslash that read its previous content has finished.
// Inside a solve the two all-reduces of every iteration guarantee that, and exchanges of the two kinds alternate
// (a rank raises the flag of exchange n+1 of the OTHER kind only after its reader of exchange n has completed).  Two
// exchanges of the SAME kind in a row with nothing in between -- lqcd_dslash called twice for the same parity, a
// solve right after such a call -- get a device-side barrier first: one generic all-reduce of a dummy value.
int peer_guard(lqcd_ctx *ctx, int kind)
{
    int rc = LQCD_OK;
    if (ctx->peer_last_kind == kind) rc = launch_peer_allreduce(ctx, &ctx->d_state->sum[3], 1, 0);
    ctx->peer_last_kind = kind;
    return rc;
}

int launch_peer_push(lqcd_ctx *ctx, const void *spinor, int parity, int gate)
{
    int rcg = peer_guard(ctx, parity);
    if (rcg) return rcg;
    dim3 grid((ctx->g.s3 + 127) / 128, 2), block(128);
#define CALL(T, L) launch_k(ctx, peer_push_kernel<T, L>, grid, block, ctx->g, (const PeerDev *)ctx->d_peer, parity, (const T *)spinor, \
                            ctx->x3_lo, ctx->x3_hi, (T)ctx->peer_sign_up, (T)ctx->peer_sign_down, (const SolverState *)ctx->d_state, gate)
    if (ctx->prec == LQCD_F64) { if (ctx->layout == 0) CALL(double, 0); else CALL(double, 1); }
    else { if (ctx->layout == 0) CALL(float, 0); else CALL(float, 1); }
#undef CALL
    int rc = lqcd_check_cuda(ctx, cudaGetLastError(), "peer push");
    return rc ? rc : peer_after_producer(ctx, parity, gate);
}

// ---- face pull: the two faces of the exchange just pushed -> the vector's own ghost slices (for consumers that are not
// the Dslash: the fermion-force kernel reads forward neighbours from the ghost slice).  Follows the push in the stream, so
// its CTA (0,0) raises the neighbours' flags like the Dslash does; every CTA waits for the rank's own two flags.
template <typename T, int LAYOUT>
__global__ void __launch_bounds__(128) peer_pull_kernel(const Geom g, const PeerDev *__restrict__ pdp, const int kind,
                                                        T *__restrict__ spinor, const int x3_lo, const int x3_hi)
{
    pdl_wait();
    pdl_trigger();
    const PeerDev &pd = *pdp;
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) peer_signal_halo(pd, kind);
    peer_wait_halo(pd, kind);
    const int up = blockIdx.y;                       // 0: ghost slice below (from down), 1: ghost slice above (from up)
    const T *__restrict__ buf = reinterpret_cast<const T *>(pd.land_self[kind][up]);
    const int x3 = up ? x3_hi : x3_lo - 1;
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= g.s3) return;
    Cx<T> p[3];
    load_vec_cg<T, LAYOUT>(buf, (size_t)g.s3, (size_t)f, (T)1, (T)0, p);
#pragma unroll
    for (int c = 0; c < 3; ++c) st_cx<T, LAYOUT, 0>(spinor, (size_t)c, (size_t)g.Vh, (size_t)x3 * g.s3 + f, p[c], L2Pol());
}

int launch_peer_pull(lqcd_ctx *ctx, void *spinor, int parity)
{
    dim3 grid((ctx->g.s3 + 127) / 128, 2), block(128);
#define CALL(T, L) launch_k(ctx, peer_pull_kernel<T, L>, grid, block, ctx->g, (const PeerDev *)ctx->d_peer, parity, (T *)spinor, ctx->x3_lo, ctx->x3_hi)
    if (ctx->prec == LQCD_F64) { if (ctx->layout == 0) CALL(double, 0); else CALL(double, 1); }
    else { if (ctx->layout == 0) CALL(float, 0); else CALL(float, 1); }
#undef CALL
    return lqcd_check_cuda(ctx, cudaGetLastError(), "peer pull");
}

// ---- generic all-reduce of up to LQCD_MAX_SHIFTS doubles, as two one-CTA kernels (publish, then gather) ----------
__global__ void peer_publish_kernel(const PeerDev *pdp, const double *vals, int nv)
{
    pdl_wait();
    pdl_trigger();
    if (threadIdx.x == 0 && blockIdx.x == 0) { peer_bump_red(*pdp, 2); __threadfence(); peer_publish(*pdp, 2, vals, nv); }
}
// out[v] = sum over ranks; which = 1: the sum is <b,b>: initialise the solver state like init_kernel's last CTA does
__global__ void peer_gather_kernel(const PeerDev *pdp, double *out, int nv, SolverState *st, int which)
{
    pdl_wait();
    pdl_trigger();
    const unsigned int n = peer_wait_red(*pdp, 2);
    if (threadIdx.x < nv) out[threadIdx.x] = peer_sum(*pdp, 2, n, threadIdx.x);
    if (which == 1 && threadIdx.x == 0) {
        const double t = peer_sum(*pdp, 2, n, 0);
        st->cur[0].rho = t;
        st->bnorm2 = t;
        if (t == 0.0) st->done = 2;
    }
}

// all-reduce nv device doubles at `vals` over the ranks, in place (nv <= LQCD_MAX_SHIFTS); which as above
int launch_peer_allreduce(lqcd_ctx *ctx, double *vals, int nv, int which)
{
    launch_k(ctx, peer_publish_kernel, dim3(1), dim3(32), (const PeerDev *)ctx->d_peer, (const double *)vals, nv);
    int rc = lqcd_check_cuda(ctx, cudaGetLastError(), "peer publish");
    if (rc || (rc = peer_phase(ctx, 1))) return rc;
    launch_k(ctx, peer_gather_kernel, dim3(1), dim3(32), (const PeerDev *)ctx->d_peer, vals, nv, ctx->d_state, which);
    return lqcd_check_cuda(ctx, cudaGetLastError(), "peer gather");
}

// ---- protocol self-test under REAL concurrency on one GPU -----------------------------------------------------
// The virtual-rank tests run the ranks in lock step (no kernel may wait for another LAUNCH on one GPU).  What they cannot
// show -- the flag / slot / counter protocol of peer.cuh with ranks that really run at the same time and really wait for
// one another -- is exercised here the way B200_PROFILING.md prescribes: ONE cooperative kernel whose CTA r plays rank r
// on its own PeerBlock (co-residency is guaranteed by the cooperative launch).  Per round, as in a CG iteration:
//   a "producer" phase   bump the counters, store a token into the two neighbours' landing buffers (kind = round & 1)
//   signal + wait_halo   then check the two tokens that arrived
//   publish + wait_red   (kind 0, then kind 1) and check the rank-ordered sum against the closed form
// with deliberately uneven delays per rank and round so that fast ranks run ahead as far as the protocol lets them.
// Any mismatch or timeout is counted.
__global__ void __launch_bounds__(128) peer_selftest_kernel(const PeerDev *pds, int rounds, unsigned int *failures, int sabotage)
{
    const PeerDev &pd = pds[blockIdx.x];
    const int P = pd.nranks, me = pd.rank, up = (me + 1) % P, down = (me + P - 1) % P;
    for (int t = 0; t < rounds; ++t) {
        // uneven pace: a rank- and round-dependent spin before each phase
        const long long pause = 200LL * ((me * 7 + t * 13) % 11);
        const long long t0 = clock64();
        while (clock64() - t0 < pause) { }
        const int kind = t & 1;
        if (threadIdx.x == 0) {
            // producer: faces = one token per direction (what a push kernel / fused push stores), then the counter
            reinterpret_cast<volatile double *>(pd.land_up[kind])[0] = 1000.0 * t + me;          // to the rank above, "from down"
            reinterpret_cast<volatile double *>(pd.land_down[kind])[0] = -(1000.0 * t + me);     // to the rank below, "from up"
            __threadfence_system();     // stands for the kernel boundary between producer and consumer
            peer_bump_halo(pd, kind);
            peer_signal_halo(pd, kind);
        }
        __syncthreads();
        if (!sabotage) peer_wait_halo(pd, kind);      // sabotage: the consumers do not wait -- the test must then FAIL
        if (threadIdx.x == 0) {
            const double a = __ldcg(reinterpret_cast<const double *>(pd.land_self[kind][0]));
            const double b = __ldcg(reinterpret_cast<const double *>(pd.land_self[kind][1]));
            if (a != 1000.0 * t + down) atomicAdd(failures, 1u);
            if (b != -(1000.0 * t + up)) atomicAdd(failures, 1u);
        }
        for (int k = 0; k < 2; ++k) {            // the two all-reduces of an iteration
            if (threadIdx.x == 0) {
                const double v = (double)((me + 1) * (t + 1) + k);
                peer_bump_red(pd, k);
                peer_publish(pd, k, &v, 1);
            }
            __syncthreads();
            // kind 0 through the generic pair (wait for all P flags, sum the slots), kind 1 the way K1 / K2 do it (own
            // value from registers, wait for the other ranks only)
            double s;
            if (k == 1 && !sabotage) s = peer_gather_with_local(pd, 1, (double)((me + 1) * (t + 1) + k));
            else {
                const unsigned int n = sabotage ? *(volatile unsigned int *)&pd.self->cnt_red[k] : peer_wait_red(pd, k);
                s = peer_sum(pd, k, n, 0);
            }
            const double want = (double)((t + 1) * (P * (P + 1) / 2) + k * P);
            if (threadIdx.x == 0 && s != want) atomicAdd(failures, 1u);
            __syncthreads();
        }
    }
    if (threadIdx.x == 0 && pd.self->timeouts) atomicAdd(failures, pd.self->timeouts);
}

extern "C" int lqcd_peer_selftest(lqcd_ctx *ctx, int nranks, int rounds, int sabotage, int *failures)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nranks < 1 || nranks > LQCD_MAX_RANKS || rounds < 1 || !failures)
        return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_peer_selftest: 1 <= nranks <= %d, rounds >= 1, failures != NULL", LQCD_MAX_RANKS);
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
    if (!coop) return lqcd_fail(ctx, LQCD_ERR_UNSUPPORTED, "lqcd_peer_selftest: no cooperative launch on this device");
    const size_t blk = align256(sizeof(PeerBlock)) + 4 * 256;       // one 256-byte "landing buffer" per (kind, direction)
    char *mem = NULL;
    PeerDev *d_pds = NULL;
    unsigned int *d_fail = NULL;
    cudaError_t e;
    if ((e = cudaMalloc(&mem, blk * nranks)) != cudaSuccess || (e = cudaMalloc(&d_pds, sizeof(PeerDev) * nranks)) != cudaSuccess ||
        (e = cudaMalloc(&d_fail, sizeof(unsigned int))) != cudaSuccess || (e = cudaMemset(mem, 0, blk * nranks)) != cudaSuccess ||
        (e = cudaMemset(d_fail, 0, sizeof(unsigned int))) != cudaSuccess) {
        cudaFree(mem); cudaFree(d_pds); cudaFree(d_fail);
        return lqcd_check_cuda(ctx, e, "lqcd_peer_selftest");
    }
    PeerDev h[LQCD_MAX_RANKS];
    memset(h, 0, sizeof(h));
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, ctx->device);
    for (int r = 0; r < nranks; ++r) {
        PeerDev &p = h[r];
        p.nranks = nranks; p.rank = r;
        p.self = (PeerBlock *)(mem + blk * r);
        for (int q = 0; q < nranks; ++q) p.peer[q] = (PeerBlock *)(mem + blk * q);
        p.up = p.peer[(r + 1) % nranks]; p.down = p.peer[(r + nranks - 1) % nranks];
        p.sign_up = p.sign_down = 1.0;
        p.wait_cycles = 3000LL * (khz > 0 ? khz : 1900000);
        for (int k = 0; k < 2; ++k) {
            for (int d = 0; d < 2; ++d) p.land_self[k][d] = (char *)p.self + align256(sizeof(PeerBlock)) + (k * 2 + d) * 256;
            p.land_up[k] = (char *)p.up + align256(sizeof(PeerBlock)) + (k * 2 + 0) * 256;
            p.land_down[k] = (char *)p.down + align256(sizeof(PeerBlock)) + (k * 2 + 1) * 256;
        }
    }
    unsigned int hf = 0;
    const PeerDev *arg_pds = d_pds;
    void *args[] = { (void *)&arg_pds, (void *)&rounds, (void *)&d_fail, (void *)&sabotage };
    if ((e = cudaMemcpy(d_pds, h, sizeof(PeerDev) * nranks, cudaMemcpyHostToDevice)) == cudaSuccess &&
        (e = cudaLaunchCooperativeKernel((const void *)peer_selftest_kernel, dim3(nranks), dim3(128), args, 0, ctx->stream)) == cudaSuccess &&
        (e = cudaStreamSynchronize(ctx->stream)) == cudaSuccess)
        e = cudaMemcpy(&hf, d_fail, sizeof(hf), cudaMemcpyDeviceToHost);
    ctx->launches++;
    cudaFree(mem); cudaFree(d_pds); cudaFree(d_fail);
    if (e != cudaSuccess) return lqcd_check_cuda(ctx, e, "lqcd_peer_selftest");
    *failures = (int)hf;
    return LQCD_OK;
}
