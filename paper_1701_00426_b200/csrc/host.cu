// host.cu -- end-to-end entry points on HOST buffers in the canonical layout (include/lqcd.h):
// host->device copy, pack, compute, unpack, device->host copy inside one blocking call.
// These are what bench.py's "e2e" figure times.  Data movement only; the arithmetic is in
// dslash.cu / solver.cu.  (the paper keeps fields resident and moves them only at
// the start and end of a Monte Carlo update; these calls are the worst case where nothing is.)
#include "common.cuh"

static int stage_reserve(lqcd_ctx *ctx, size_t bytes)
{
    if (ctx->stage_bytes >= bytes) return LQCD_OK;
    if (ctx->stage) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->stage); ctx->stage = NULL; ctx->stage_bytes = 0; }
    int rc = lqcd_check_cuda(ctx, cudaMalloc(&ctx->stage, bytes), "staging cudaMalloc");
    if (rc) return rc;
    ctx->stage_bytes = bytes;
    return LQCD_OK;
}

static size_t up256(size_t b) { return (b + 255) & ~(size_t)255; }

extern "C" int lqcd_dslash_host(lqcd_ctx *ctx, int parity, void *out_host, const void *in_host, const void *links_host)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!out_host || !in_host || !links_host) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host: null pointer");
    if (parity != 0 && parity != 1) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host: parity %d", parity);
    const size_t Vh = (size_t)ctx->g.Vh;
    const size_t canon_links = Vh * 2 * 4 * 9 * 16, canon_sp = Vh * 3 * 16;
    const size_t nat_links = up256(lqcd_links_bytes(ctx)), nat_sp = up256(lqcd_spinor_bytes(ctx));
    if ((rc = stage_reserve(ctx, up256(canon_links) + up256(canon_sp) + nat_links + 2 * nat_sp))) return rc;
    char *c_links = (char *)ctx->stage, *c_sp = c_links + up256(canon_links);
    char *n_links = c_sp + up256(canon_sp), *n_in = n_links + nat_links, *n_out = n_in + nat_sp;
    cudaStream_t s = ctx->stream;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_links, links_host, canon_links, cudaMemcpyHostToDevice, s), "H2D links"))) return rc;
    if ((rc = lqcd_pack_links(ctx, n_links, c_links))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_sp, in_host, canon_sp, cudaMemcpyHostToDevice, s), "H2D spinor"))) return rc;
    if ((rc = lqcd_pack_spinor(ctx, 1 - parity, n_in, c_sp))) return rc;
    if ((rc = lqcd_dslash(ctx, parity, n_out, n_in, n_links))) return rc;
    if ((rc = lqcd_unpack_spinor(ctx, parity, c_sp, n_out))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(out_host, c_sp, canon_sp, cudaMemcpyDeviceToHost, s), "D2H spinor"))) return rc;
    return lqcd_check_cuda(ctx, cudaStreamSynchronize(s), "lqcd_dslash_host");
}

// As lqcd_dslash_host, but the link field is already resident in native form (uploaded and packed once
// per gauge configuration, as the paper does: PAPER.md:276); only the vectors cross the bus.
extern "C" int lqcd_dslash_host_vectors(lqcd_ctx *ctx, int parity, void *out_host, const void *in_host,
                                        const void *links_native_dev)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!out_host || !in_host || !links_native_dev) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host_vectors: null pointer");
    if (parity != 0 && parity != 1) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host_vectors: parity %d", parity);
    const size_t canon_sp = (size_t)ctx->g.Vh * 3 * 16;
    const size_t nat_sp = up256(lqcd_spinor_bytes(ctx));
    if ((rc = stage_reserve(ctx, up256(canon_sp) + 2 * nat_sp))) return rc;
    char *c_sp = (char *)ctx->stage, *n_in = c_sp + up256(canon_sp), *n_out = n_in + nat_sp;
    cudaStream_t s = ctx->stream;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_sp, in_host, canon_sp, cudaMemcpyHostToDevice, s), "H2D spinor"))) return rc;
    if ((rc = lqcd_pack_spinor(ctx, 1 - parity, n_in, c_sp))) return rc;
    if ((rc = lqcd_dslash(ctx, parity, n_out, n_in, links_native_dev))) return rc;
    if ((rc = lqcd_unpack_spinor(ctx, parity, c_sp, n_out))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(out_host, c_sp, canon_sp, cudaMemcpyDeviceToHost, s), "D2H spinor"))) return rc;
    return lqcd_check_cuda(ctx, cudaStreamSynchronize(s), "lqcd_dslash_host_vectors");
}

extern "C" int lqcd_cg_multishift_host(lqcd_ctx *ctx, int nshift, const double *shifts, const void *rhs_host,
                                       void *solutions_host, const void *links_host, double mass, double tol,
                                       int max_iter, int *iters, int *conv_iter, double *rel_resid)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return lqcd_fail(ctx, LQCD_ERR_ARG, "nshift %d not in [1,%d]", nshift, LQCD_MAX_SHIFTS);
    if (!rhs_host || !solutions_host || !links_host || !shifts) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_cg_multishift_host: null pointer");
    const size_t Vh = (size_t)ctx->g.Vh;
    const size_t canon_links = Vh * 2 * 4 * 9 * 16, canon_sp = Vh * 3 * 16;
    const size_t nat_links = up256(lqcd_links_bytes(ctx)), nat_sp = up256(lqcd_spinor_bytes(ctx));
    const size_t ws = up256(lqcd_workspace_bytes(ctx, nshift));
    if ((rc = stage_reserve(ctx, up256(canon_links) + up256(canon_sp) + nat_links + (size_t)(1 + nshift) * nat_sp + ws))) return rc;
    char *c_links = (char *)ctx->stage, *c_sp = c_links + up256(canon_links);
    char *n_links = c_sp + up256(canon_sp), *n_b = n_links + nat_links, *n_x = n_b + nat_sp;
    char *wsp = n_x + (size_t)nshift * nat_sp;
    void *old_ws = ctx->ws; size_t old_ws_bytes = ctx->ws_bytes;
    cudaStream_t s = ctx->stream;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_links, links_host, canon_links, cudaMemcpyHostToDevice, s), "H2D links"))) return rc;
    if ((rc = lqcd_pack_links(ctx, n_links, c_links))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_sp, rhs_host, canon_sp, cudaMemcpyHostToDevice, s), "H2D rhs"))) return rc;
    if ((rc = lqcd_pack_spinor(ctx, LQCD_EVEN, n_b, c_sp))) return rc;
    void *xs[LQCD_MAX_SHIFTS];
    for (int i = 0; i < nshift; ++i) xs[i] = n_x + (size_t)i * nat_sp;
    ctx->ws = wsp; ctx->ws_bytes = ws;
    int solve_rc = lqcd_cg_multishift(ctx, nshift, shifts, n_b, xs, n_links, mass, tol, max_iter, iters, conv_iter, rel_resid);
    ctx->ws = old_ws; ctx->ws_bytes = old_ws_bytes;
    if (solve_rc != LQCD_OK && solve_rc != LQCD_ERR_NOT_CONVERGED) return solve_rc;
    for (int i = 0; i < nshift; ++i) {
        if ((rc = lqcd_unpack_spinor(ctx, LQCD_EVEN, c_sp, xs[i]))) return rc;
        if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync((char *)solutions_host + (size_t)i * canon_sp, c_sp, canon_sp, cudaMemcpyDeviceToHost, s), "D2H solution"))) return rc;
    }
    if ((rc = lqcd_check_cuda(ctx, cudaStreamSynchronize(s), "lqcd_cg_multishift_host"))) return rc;
    return solve_rc;
}
