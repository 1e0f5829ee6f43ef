// api.cu -- context management, argument checking and the host-buffer entry points of the
// C ABI declared in include/lqcd.h.  No arithmetic of the method lives here.
#include <stdarg.h>
#include <stdlib.h>

#include "common.cuh"

static thread_local char g_create_err[256] = "";
static void clear_l2_window(lqcd_ctx *ctx);
static void apply_l2_window(lqcd_ctx *ctx);

extern "C" const char *lqcd_version(void) { return "lqcd_b200 0.1 (sm_100a)"; }

int lqcd_fail(lqcd_ctx *ctx, int code, const char *fmt, ...)
{
    char *dst = ctx ? ctx->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 256, fmt, ap);
    va_end(ap);
    return code;
}

int lqcd_check_cuda(lqcd_ctx *ctx, cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return LQCD_OK;
    return lqcd_fail(ctx, LQCD_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

size_t elem_size(const lqcd_ctx *ctx) { return ctx->prec == LQCD_F64 ? 8 : 4; }

extern "C" const char *lqcd_last_error(const lqcd_ctx *ctx) { return ctx ? ctx->err : g_create_err; }

extern "C" int lqcd_create(lqcd_ctx **out, const int dims[4], int prec, int recon,
                           int antiperiodic_t, int device, void *cuda_stream)
{
    if (!out) return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: ctx is NULL");
    *out = NULL;
    if (!dims) return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: dims is NULL");
    long long V = 1;
    for (int i = 0; i < 4; ++i) {
        if (dims[i] < 2 || (dims[i] & 1))
            return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: dims[%d] = %d must be even and >= 2", i, dims[i]);
        V *= dims[i];
        if (V >= (1LL << 31)) return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: volume must be < 2^31");
    }
    if (prec != LQCD_F64 && prec != LQCD_F32) return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: bad prec %d", prec);
    if (recon != LQCD_RECON_18 && recon != LQCD_RECON_12)
        return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: bad recon %d", recon);
    if (antiperiodic_t != 0 && antiperiodic_t != 1)
        return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: antiperiodic_t must be 0 or 1");
    if (device < 0) return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: bad device %d", device);

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return lqcd_fail(NULL, LQCD_ERR_CUDA, "lqcd_create: no CUDA device (%s); there is no CPU fallback",
                         cudaGetErrorString(e));
    if (device >= ndev) return lqcd_fail(NULL, LQCD_ERR_ARG, "lqcd_create: device %d of %d", device, ndev);
    if ((e = cudaSetDevice(device)) != cudaSuccess) return lqcd_check_cuda(NULL, e, "cudaSetDevice");

    lqcd_ctx *c = (lqcd_ctx *)calloc(1, sizeof(lqcd_ctx));
    if (!c) return lqcd_fail(NULL, LQCD_ERR_CUDA, "lqcd_create: out of host memory");
    Geom &g = c->g;
    g.N0 = dims[0]; g.N1 = dims[1]; g.N2 = dims[2]; g.N3 = dims[3];
    g.Nh0 = g.N0 / 2;
    g.Vh = (int)(V / 2);
    g.Ls = g.Vh;
    g.s1 = g.Nh0; g.s2 = g.Nh0 * g.N1; g.s3 = g.Nh0 * g.N1 * g.N2;
    g.ap = antiperiodic_t;
    g.dNh0 = make_fastdiv((uint32_t)g.Nh0);
    g.dN1 = make_fastdiv((uint32_t)g.N1);
    g.dN2 = make_fastdiv((uint32_t)g.N2);
    c->prec = prec; c->recon = recon; c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->layout = 0;
    c->dslash_block = 128;
    c->dslash_minblocks = 0;   // 0: the per-precision default of dslash.cu
    c->blas_block = 256;
    c->blas_ctas_per_sm = 8;
    c->poll_chunk = 8;
    c->pdl = 1;
    c->graph = 1;
    c->dslash_persist = 0;
    c->iter_mask = 15;
    c->staples_variant = 2;
    c->force_stage = 1;
    c->force_block = 8;    // measured at 32^4 fp64, 8 shifts: whole force 1.13 ms (one Dslash per shift), 0.65 (blocks of 4), 0.55 (one block of 8)
    c->staples_x2block = 4;
    c->peer_wait_ms = 3000;
    c->launch_stream = c->stream;
    c->x3_lo = 0;
    c->x3_hi = g.N3;
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) { free(c); return lqcd_check_cuda(NULL, e, "cudaGetDeviceProperties"); }
    c->num_sms = prop.multiProcessorCount;
    c->max_partials = g.Vh / 32 + 1024;   // >= the largest grid any reducing kernel uses
    if ((e = cudaMalloc(&c->d_state, sizeof(SolverState))) != cudaSuccess ||
        (e = cudaMalloc(&c->d_partials, sizeof(double) * 2 * c->max_partials)) != cudaSuccess ||
        (e = cudaMallocHost(&c->h_flag, 64)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev[0], cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev[1], cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking)) != cudaSuccess ||
        (e = cudaMemset(c->d_state, 0, sizeof(SolverState))) != cudaSuccess) {
        int rc = lqcd_check_cuda(NULL, e, "lqcd_create: allocating solver state");
        cudaFree(c->d_state); cudaFree(c->d_partials); if (c->h_flag) cudaFreeHost(c->h_flag);
        if (c->ev[0]) cudaEventDestroy(c->ev[0]);
        if (c->ev[1]) cudaEventDestroy(c->ev[1]);
        if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
        free(c);
        return rc;
    }
    *out = c;
    return LQCD_OK;
}

extern "C" int lqcd_destroy(lqcd_ctx *ctx)
{
    if (!ctx) return LQCD_ERR_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    clear_l2_window(ctx);
    lqcd_peer_destroy(ctx);
    cudaFree(ctx->d_state);
    cudaFree(ctx->d_partials);
    cudaFreeHost(ctx->h_flag);
    cudaEventDestroy(ctx->ev[0]);
    cudaEventDestroy(ctx->ev[1]);
    cudaFree(ctx->stage);
    if (ctx->h2d_stream) cudaStreamDestroy(ctx->h2d_stream);
    if (ctx->d2h_stream) cudaStreamDestroy(ctx->d2h_stream);
    for (int k = 0; k < 3; ++k) for (int j = 0; j < 2; ++j) if (ctx->pipe_ev[k][j]) cudaEventDestroy(ctx->pipe_ev[k][j]);
    if (ctx->chunk_exec) cudaGraphExecDestroy(ctx->chunk_exec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    free(ctx);
    return LQCD_OK;
}

struct OptDesc { const char *name; size_t off; long lo, hi; };
#define OPT(field, lo, hi) { #field, offsetof(lqcd_ctx, field), lo, hi }
static const OptDesc g_opts[] = {
    OPT(layout, 0, 1), OPT(l2_hints, 0, 1), OPT(l2_persist, 0, 4), OPT(link_pad, 0, 1 << 20), OPT(dslash_block, 32, 256), OPT(dslash_minblocks, 0, 4),
    OPT(blas_block, 64, 256), OPT(blas_ctas_per_sm, 1, 32), OPT(poll_chunk, 1, 1024),
    OPT(pdl, 0, 1), OPT(graph, 0, 1), OPT(dslash_persist, 0, 16), OPT(iter_mask, 0, 15), OPT(staples_variant, 0, 2), OPT(staples_minblocks, 0, 4), OPT(peer_wait_ms, 0, 600000), OPT(force_stage, 0, 1), OPT(force_block, 0, 8), OPT(staples_x2block, 0, 64), OPT(backfield_format, 0, 1),
};

extern "C" int lqcd_set_option(lqcd_ctx *ctx, const char *name, long value)
{
    if (!ctx || !name) return LQCD_ERR_ARG;
    for (const OptDesc &o : g_opts) {
        if (strcmp(o.name, name)) continue;
        if (value < o.lo || value > o.hi) return lqcd_fail(ctx, LQCD_ERR_ARG, "option %s: %ld out of [%ld,%ld]", name, value, o.lo, o.hi);
        if (!strcmp(name, "layout") && ctx->layout_locked && value != ctx->layout)
            return lqcd_fail(ctx, LQCD_ERR_ARG, "option layout: fields were already packed in layout %d", ctx->layout);
        if ((!strcmp(name, "dslash_block") || !strcmp(name, "blas_block")) && (value % 32))
            return lqcd_fail(ctx, LQCD_ERR_ARG, "option %s must be a multiple of 32", name);
        if (!strcmp(name, "backfield_format") && ctx->backfield_locked && value != ctx->backfield_format)
            return lqcd_fail(ctx, LQCD_ERR_ARG, "option backfield_format: a backfield was already packed in format %d", ctx->backfield_format);
        if (!strcmp(name, "link_pad")) {
            if (ctx->layout_locked && value != ctx->link_pad) return lqcd_fail(ctx, LQCD_ERR_ARG, "option link_pad: fields were already packed");
            if (value % 8) return lqcd_fail(ctx, LQCD_ERR_ARG, "option link_pad must be a multiple of 8 sites");
        }
        *(int *)((char *)ctx + o.off) = (int)value;
        if (!strcmp(name, "l2_persist")) apply_l2_window(ctx);     // takes effect (or is undone) at once
        ctx->g.Ls = ctx->g.Vh + ctx->link_pad;   // link plane stride in sites
        return LQCD_OK;
    }
    return lqcd_fail(ctx, LQCD_ERR_ARG, "unknown option %s", name);
}

extern "C" long lqcd_get_option(const lqcd_ctx *ctx, const char *name)
{
    if (!ctx || !name) return -1;
    if (!strcmp(name, "launches")) return ctx->launches;
    if (!strcmp(name, "num_sms")) return ctx->num_sms;
    if (!strcmp(name, "graph_active")) return ctx->graph_active;
    if (!strcmp(name, "peer_timeouts")) return peer_timeouts((lqcd_ctx *)ctx);
    if (!strcmp(name, "staples_ran")) return ctx->staples_ran;
    if (!strcmp(name, "l2_window_bytes")) return ctx->l2_window_bytes;
    if (!strcmp(name, "l2_max_persist")) return ctx->l2_max_persist;
    for (const OptDesc &o : g_opts)
        if (!strcmp(o.name, name)) return *(const int *)((const char *)ctx + o.off);
    return -1;
}

extern "C" size_t lqcd_spinor_bytes(const lqcd_ctx *ctx)
{
    return ctx ? (size_t)ctx->g.Vh * 6 * elem_size(ctx) : 0;
}

extern "C" size_t lqcd_links_bytes(const lqcd_ctx *ctx)
{
    if (!ctx) return 0;
    size_t rows = ctx->recon == LQCD_RECON_12 ? 2 : 3;
    return (size_t)ctx->g.Ls * 2 * 4 * rows * 3 * 2 * elem_size(ctx);
}

// workspace = tmp_o, q, r, p  +  one p_i per shift (the base shift's is unused but keeps indexing
// simple) ; each rounded up to 256 bytes.
static size_t vec_stride(const lqcd_ctx *ctx) { return (lqcd_spinor_bytes(ctx) + 255) & ~(size_t)255; }

extern "C" size_t lqcd_workspace_bytes(const lqcd_ctx *ctx, int nshift)
{
    if (!ctx || nshift < 1 || nshift > LQCD_MAX_SHIFTS) return 0;
    return vec_stride(ctx) * (size_t)(4 + nshift);
}

// Optional (option l2_persist): ask the driver to keep the four vectors every CG iteration re-reads
// (tmp_o, q, r, p: the head of the workspace) in the persisting part of L2 while links stream by.
// Undo apply_l2_window: the access-policy window is an attribute of the (possibly shared) stream and the
// persisting lines belong to the device, so both must be cleared when the option is switched off or the
// context goes away -- otherwise later work on the same stream inherits a window over freed memory.
static void clear_l2_window(lqcd_ctx *ctx)
{
    if (!ctx->l2_window_bytes) return;
    cudaStreamAttrValue v;
    memset(&v, 0, sizeof(v));
    v.accessPolicyWindow.num_bytes = 0;
    v.accessPolicyWindow.hitProp = cudaAccessPropertyNormal;
    v.accessPolicyWindow.missProp = cudaAccessPropertyNormal;
    // put back what apply_l2_window found (the stream may be shared and the carve-out is device-wide: other
    // contexts or frameworks may have set their own)
    if (ctx->l2_saved) v = ctx->l2_prev_attr;
    if (cudaStreamSetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &v) != cudaSuccess) cudaGetLastError();
    // a persisting-L2 limit left at its maximum keeps 2/3 of the L2 away from every later kernel of the
    // process (measured: CG at 32^3 x 8 89.8 instead of 64 us per iteration): restore the previous limit.
    // Lines of OUR window that are still marked persisting are demoted only when nobody else had a
    // carve-out (previous limit 0); otherwise they age out by themselves.
    if (ctx->l2_saved && ctx->l2_prev_limit == 0 && cudaCtxResetPersistingL2Cache() != cudaSuccess) cudaGetLastError();
    if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, ctx->l2_saved ? ctx->l2_prev_limit : 0) != cudaSuccess) cudaGetLastError();
    ctx->l2_saved = 0;
    ctx->l2_window_bytes = 0;
}

static void apply_l2_window(lqcd_ctx *ctx)
{
    clear_l2_window(ctx);
    if (!ctx->l2_persist || !ctx->ws) return;
    int max_persist = 0, max_window = 0;
    cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, ctx->device);
    cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, ctx->device);
    // 1: 4 vectors, misses streaming; 2: 3 vectors (fits the carve-out), misses normal;
    // 3: 4 vectors, misses normal; 4: 2 vectors, misses normal
    int nvec = ctx->l2_persist == 2 ? 3 : (ctx->l2_persist == 4 ? 2 : 4);
    size_t want = vec_stride(ctx) * nvec;
    if (want > ctx->ws_bytes) want = ctx->ws_bytes;
    size_t win = want < (size_t)max_window ? want : (size_t)max_window;
    if (max_persist <= 0 || win == 0) return;
    // remember the device limit and the stream's window as we found them (restored by clear_l2_window)
    ctx->l2_prev_limit = 0;
    memset(&ctx->l2_prev_attr, 0, sizeof(ctx->l2_prev_attr));
    if (cudaDeviceGetLimit(&ctx->l2_prev_limit, cudaLimitPersistingL2CacheSize) != cudaSuccess) { cudaGetLastError(); ctx->l2_prev_limit = 0; }
    if (cudaStreamGetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &ctx->l2_prev_attr) != cudaSuccess) {
        cudaGetLastError();
        memset(&ctx->l2_prev_attr, 0, sizeof(ctx->l2_prev_attr));
    }
    ctx->l2_saved = 1;
    if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)max_persist) != cudaSuccess) { cudaGetLastError(); ctx->l2_saved = 0; return; }
    cudaStreamAttrValue v;
    memset(&v, 0, sizeof(v));
    v.accessPolicyWindow.base_ptr = ctx->ws;
    v.accessPolicyWindow.num_bytes = win;
    v.accessPolicyWindow.hitRatio = win <= (size_t)max_persist ? 1.0f : (float)max_persist / (float)win;
    v.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    v.accessPolicyWindow.missProp = ctx->l2_persist == 1 ? cudaAccessPropertyStreaming : cudaAccessPropertyNormal;
    if (cudaStreamSetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &v) != cudaSuccess) {
        cudaGetLastError();
        if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, ctx->l2_prev_limit) != cudaSuccess) cudaGetLastError();
        ctx->l2_saved = 0;
        return;
    }
    ctx->l2_window_bytes = (long)win;
    ctx->l2_max_persist = max_persist;
}

extern "C" int lqcd_set_workspace(lqcd_ctx *ctx, void *dev_ptr, size_t bytes)
{
    if (!ctx) return LQCD_ERR_ARG;
    if (!dev_ptr || ((uintptr_t)dev_ptr & 15)) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_set_workspace: null or unaligned pointer");
    if (bytes < lqcd_workspace_bytes(ctx, 1)) return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "lqcd_set_workspace: %zu bytes < minimum %zu", bytes, lqcd_workspace_bytes(ctx, 1));
    ctx->ws = dev_ptr;
    ctx->ws_bytes = bytes;
    apply_l2_window(ctx);
    return LQCD_OK;
}

void *ws_vec(lqcd_ctx *ctx, int k) { return (char *)ctx->ws + vec_stride(ctx) * (size_t)k; }

// ---- thin checked wrappers ------------------------------------------------------------------
#define REQUIRE(cond, ...) do { if (!(cond)) return lqcd_fail(ctx, LQCD_ERR_ARG, __VA_ARGS__); } while (0)

static int enter(lqcd_ctx *ctx)
{
    if (!ctx) return LQCD_ERR_ARG;
    return lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
}

extern "C" int lqcd_pack_links(lqcd_ctx *ctx, void *native_dev, const void *canonical_dev)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(native_dev && canonical_dev, "lqcd_pack_links: null pointer");
    ctx->layout_locked = 1;
    return launch_pack_links(ctx, native_dev, canonical_dev);
}

extern "C" int lqcd_pack_spinor(lqcd_ctx *ctx, int parity, void *native_dev, const void *canonical_dev)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(native_dev && canonical_dev, "lqcd_pack_spinor: null pointer");
    REQUIRE(parity == 0 || parity == 1, "lqcd_pack_spinor: parity %d", parity);
    ctx->layout_locked = 1;
    return launch_pack_spinor(ctx, parity, native_dev, canonical_dev);
}

extern "C" int lqcd_unpack_spinor(lqcd_ctx *ctx, int parity, void *canonical_dev, const void *native_dev)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(native_dev && canonical_dev, "lqcd_unpack_spinor: null pointer");
    REQUIRE(parity == 0 || parity == 1, "lqcd_unpack_spinor: parity %d", parity);
    return launch_unpack_spinor(ctx, parity, canonical_dev, native_dev);
}

extern "C" int lqcd_dslash(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(out && in && links, "lqcd_dslash: null pointer");
    REQUIRE(parity == 0 || parity == 1, "lqcd_dslash: parity %d", parity);
    REQUIRE(out != in, "lqcd_dslash: out and in alias");
    if (ctx->peer_on && (rc = launch_peer_push(ctx, in, 1 - parity, 0))) return rc;     // faces of `in` to the neighbours
    return launch_dslash(ctx, parity, out, in, links, NULL, 0.0, 0, 0);
}

extern "C" int lqcd_dslash_multi(lqcd_ctx *ctx, int parity, int n, void *const *outs, const void *const *ins, const void *links)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(outs && ins && links, "lqcd_dslash_multi: null pointer");
    REQUIRE(parity == 0 || parity == 1, "lqcd_dslash_multi: parity %d", parity);
    REQUIRE(n >= 1 && n <= LQCD_MAX_SHIFTS, "lqcd_dslash_multi: n = %d not in [1,%d]", n, LQCD_MAX_SHIFTS);
    for (int r = 0; r < n; ++r) {
        REQUIRE(outs[r] && ins[r], "lqcd_dslash_multi: vector %d is null", r);
        for (int q = 0; q < n; ++q) REQUIRE(outs[r] != ins[q], "lqcd_dslash_multi: output %d aliases input %d", r, q);
    }
    if (ctx->backfield || ctx->peer_on || ctx->halo_fn || ctx->x3_lo != 0 || ctx->x3_hi != ctx->g.N3)
        return lqcd_fail(ctx, LQCD_ERR_UNSUPPORTED, "lqcd_dslash_multi: plain contexts only (no backfield, no slab); use lqcd_dslash");
    return launch_dslash_multi(ctx, parity, n, outs, ins, links, ctx->force_block >= 8 ? 8 : 4);
}

extern "C" size_t lqcd_backfield_bytes(const lqcd_ctx *ctx)
{
    return ctx ? (size_t)ctx->g.Vh * 2 * 4 * elem_size(ctx) * (ctx->backfield_format ? 2 : 1) : 0;
}

extern "C" int lqcd_pack_backfield(lqcd_ctx *ctx, void *native_dev, const void *canonical_dev)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(native_dev && canonical_dev, "lqcd_pack_backfield: null pointer");
    ctx->backfield_locked = 1;
    return launch_pack_backfield(ctx, native_dev, canonical_dev);
}

extern "C" int lqcd_set_backfield(lqcd_ctx *ctx, const void *backfield_native_dev)
{
    if (!ctx) return LQCD_ERR_ARG;
    REQUIRE(!((uintptr_t)backfield_native_dev & 15), "lqcd_set_backfield: pointer not 16-byte aligned");
    ctx->backfield = backfield_native_dev;
    return LQCD_OK;
}

extern "C" int lqcd_dslash_backfield(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                                     const void *backfield)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(out && in && links && backfield, "lqcd_dslash_backfield: null pointer");
    REQUIRE(parity == 0 || parity == 1, "lqcd_dslash_backfield: parity %d", parity);
    REQUIRE(out != in, "lqcd_dslash_backfield: out and in alias");
    // peer transport: the faces of `in` go to the neighbours first, exactly as in lqcd_dslash (the kernel that follows
    // raises the flags and reads the landing buffers; without the push it would find the flags of the PREVIOUS
    // exchange already raised and read stale faces)
    if (ctx->peer_on && (rc = launch_peer_push(ctx, in, 1 - parity, 0))) return rc;
    const void *saved = ctx->backfield;
    ctx->backfield = backfield;
    rc = launch_dslash(ctx, parity, out, in, links, NULL, 0.0, 0, 0);
    ctx->backfield = saved;
    return rc;
}

extern "C" int lqcd_dslash_slices(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                                  int x3_lo, int x3_hi)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(out && in && links, "lqcd_dslash_slices: null pointer");
    REQUIRE(parity == 0 || parity == 1, "lqcd_dslash_slices: parity %d", parity);
    REQUIRE(out != in, "lqcd_dslash_slices: out and in alias");
    REQUIRE(0 <= x3_lo && x3_lo < x3_hi && x3_hi <= ctx->g.N3, "lqcd_dslash_slices: bad slice range [%d,%d)", x3_lo, x3_hi);
    return launch_dslash(ctx, parity, out, in, links, NULL, 0.0, 0, 0, x3_lo, x3_hi);
}

extern "C" size_t lqcd_halo_bytes(const lqcd_ctx *ctx)
{
    return ctx ? (size_t)ctx->g.s3 * 6 * elem_size(ctx) : 0;
}

extern "C" int lqcd_halo_pack(lqcd_ctx *ctx, void *buf, const void *spinor, int x3, double sign)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(buf && spinor, "lqcd_halo_pack: null pointer");
    REQUIRE(0 <= x3 && x3 < ctx->g.N3, "lqcd_halo_pack: slice %d", x3);
    return launch_halo(ctx, 1, buf, (void *)spinor, x3, sign);
}

extern "C" int lqcd_halo_unpack(lqcd_ctx *ctx, void *spinor, const void *buf, int x3)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(buf && spinor, "lqcd_halo_unpack: null pointer");
    REQUIRE(0 <= x3 && x3 < ctx->g.N3, "lqcd_halo_unpack: slice %d", x3);
    return launch_halo(ctx, 0, (void *)buf, spinor, x3, 1.0);
}

extern "C" int lqcd_halo_pack_faces(lqcd_ctx *ctx, void *buf_top, void *buf_bottom, const void *spinor,
                                    double sign_top, double sign_bottom)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(buf_top && buf_bottom && spinor, "lqcd_halo_pack_faces: null pointer");
    return launch_halo2(ctx, 1, buf_top, buf_bottom, (void *)spinor, ctx->x3_hi - 1, ctx->x3_lo, sign_top, sign_bottom);
}

extern "C" int lqcd_halo_unpack_ghosts(lqcd_ctx *ctx, void *spinor, const void *buf_from_down, const void *buf_from_up)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(buf_from_down && buf_from_up && spinor, "lqcd_halo_unpack_ghosts: null pointer");
    REQUIRE(ctx->x3_lo >= 1 && ctx->x3_hi < ctx->g.N3, "lqcd_halo_unpack_ghosts: the context has no ghost slices");
    return launch_halo2(ctx, 0, (void *)buf_from_down, (void *)buf_from_up, spinor, ctx->x3_lo - 1, ctx->x3_hi, 1.0, 1.0);
}

extern "C" int lqcd_set_slab(lqcd_ctx *ctx, int x3_lo, int x3_hi, int solve_parity, lqcd_halo_fn halo,
                             lqcd_allreduce_fn allreduce, void *user)
{
    int rc = enter(ctx); if (rc) return rc;
    // every argument is validated before any field of the context changes
    REQUIRE(solve_parity == 0 || solve_parity == 1, "lqcd_set_slab: solve_parity %d", solve_parity);
    REQUIRE(0 <= x3_lo && x3_lo < x3_hi && x3_hi <= ctx->g.N3, "lqcd_set_slab: bad slice range [%d,%d)", x3_lo, x3_hi);
    REQUIRE((halo == NULL) == (allreduce == NULL), "lqcd_set_slab: give both hooks or neither");
    REQUIRE(!ctx->peer_mem, "lqcd_set_slab: the context uses the peer transport (lqcd_peer_init); call lqcd_peer_disconnect first");
    ctx->solve_parity = solve_parity;
    ctx->x3_lo = x3_lo; ctx->x3_hi = x3_hi;
    ctx->halo_fn = halo; ctx->allreduce_fn = allreduce; ctx->comm_user = user;
    if (ctx->chunk_exec) { cudaGraphExecDestroy(ctx->chunk_exec); ctx->chunk_exec = NULL; }
    return LQCD_OK;
}

extern "C" int lqcd_mdagm(lqcd_ctx *ctx, void *out_e, const void *in_e, const void *links, double mass, double sigma)
{
    int rc = enter(ctx); if (rc) return rc;
    REQUIRE(out_e && in_e && links, "lqcd_mdagm: null pointer");
    REQUIRE(out_e != in_e, "lqcd_mdagm: out and in alias");
    if (!ctx->ws) return lqcd_fail(ctx, LQCD_ERR_WORKSPACE, "lqcd_mdagm: no workspace set");
    void *tmp_o = ws_vec(ctx, 0);
    const int par = ctx->solve_parity;     // LQCD_EVEN unless a slab says otherwise
    if (ctx->peer_on) { if ((rc = launch_peer_push(ctx, in_e, par, 0))) return rc; }
    else if (ctx->halo_fn && ctx->halo_fn(ctx->comm_user, (void *)in_e, par)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "halo hook failed");
    rc = launch_dslash(ctx, 1 - par, tmp_o, in_e, links, NULL, 0.0, 0, 0);
    if (rc) return rc;
    if (ctx->peer_on) { if ((rc = launch_peer_push(ctx, tmp_o, 1 - par, 0))) return rc; }
    else if (ctx->halo_fn && ctx->halo_fn(ctx->comm_user, tmp_o, 1 - par)) return lqcd_fail(ctx, LQCD_ERR_CUDA, "halo hook failed");
    return launch_dslash(ctx, par, out_e, tmp_o, links, in_e, mass * mass + sigma, 0, 0);
}
