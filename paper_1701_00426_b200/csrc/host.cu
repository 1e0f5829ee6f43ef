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

// n applications out[j] = D in[j] on host vectors, links resident, as ONE pipelined call: application j's
// upload (h2d_stream), its pack -> Dslash -> unpack (the context's stream) and its download (d2h_stream) are
// chained by events, canonical staging is double-buffered, so the download of application j runs while
// application j+1 is uploaded (PCIe is full duplex) and computed.
extern "C" int lqcd_dslash_host_vectors_batch(lqcd_ctx *ctx, int n, const int *parities, void *const *outs_host,
                                              const void *const *ins_host, const void *links_native_dev)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (n < 1 || !parities || !outs_host || !ins_host || !links_native_dev)
        return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host_vectors_batch: null pointer or n < 1");
    for (int j = 0; j < n; ++j) {
        if (!outs_host[j] || !ins_host[j]) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host_vectors_batch: vector %d is null", j);
        if (parities[j] != 0 && parities[j] != 1) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_dslash_host_vectors_batch: parity %d", parities[j]);
    }
    if (!ctx->h2d_stream) {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->h2d_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking);
        for (int k = 0; k < 3 && e == cudaSuccess; ++k)
            for (int j = 0; j < 2 && e == cudaSuccess; ++j) e = cudaEventCreateWithFlags(&ctx->pipe_ev[k][j], cudaEventDisableTiming);
        if (e != cudaSuccess) return lqcd_check_cuda(ctx, e, "copy pipeline setup");
    }
    const size_t canon_sp = (size_t)ctx->g.Vh * 3 * 16, csp = up256(canon_sp);
    const size_t nat_sp = up256(lqcd_spinor_bytes(ctx));
    if ((rc = stage_reserve(ctx, 4 * csp + 2 * nat_sp))) return rc;
    char *c_in[2] = { (char *)ctx->stage, (char *)ctx->stage + csp };
    char *c_out[2] = { (char *)ctx->stage + 2 * csp, (char *)ctx->stage + 3 * csp };
    char *n_in = (char *)ctx->stage + 4 * csp, *n_out = n_in + nat_sp;
    cudaStream_t s = ctx->stream, up = ctx->h2d_stream, dn = ctx->d2h_stream;
    cudaEvent_t(*ev)[2] = ctx->pipe_ev;
    // whatever the caller enqueued on the context's stream before this call comes first
    if ((rc = lqcd_check_cuda(ctx, cudaEventRecord(ev[1][0], s), "pipeline fence"))) return rc;
    cudaStreamWaitEvent(up, ev[1][0], 0);
    for (int j = 0; j < n; ++j) {
        const int sl = j & 1;
        if (j >= 2) cudaStreamWaitEvent(up, ev[1][sl], 0);              // pack of j-2 has read c_in[sl]
        if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_in[sl], ins_host[j], canon_sp, cudaMemcpyHostToDevice, up), "H2D spinor"))) return rc;
        cudaEventRecord(ev[0][sl], up);
        cudaStreamWaitEvent(s, ev[0][sl], 0);
        if (j >= 2) cudaStreamWaitEvent(s, ev[2][sl], 0);               // download of j-2 has read c_out[sl]
        if ((rc = lqcd_pack_spinor(ctx, 1 - parities[j], n_in, c_in[sl]))) return rc;
        if ((rc = lqcd_dslash(ctx, parities[j], n_out, n_in, links_native_dev))) return rc;
        if ((rc = lqcd_unpack_spinor(ctx, parities[j], c_out[sl], n_out))) return rc;
        cudaEventRecord(ev[1][sl], s);
        cudaStreamWaitEvent(dn, ev[1][sl], 0);
        if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(outs_host[j], c_out[sl], canon_sp, cudaMemcpyDeviceToHost, dn), "D2H spinor"))) return rc;
        cudaEventRecord(ev[2][sl], dn);
    }
    // later work on the context's stream is ordered after the last download
    cudaStreamWaitEvent(s, ev[2][(n - 1) & 1], 0);
    if ((rc = lqcd_check_cuda(ctx, cudaStreamSynchronize(dn), "lqcd_dslash_host_vectors_batch"))) return rc;
    return lqcd_check_cuda(ctx, cudaStreamSynchronize(s), "lqcd_dslash_host_vectors_batch");
}

// As lqcd_cg_multishift_host with the link field resident in native form: the right-hand side goes up, the
// nshift solutions come down, and the 10^2-10^3 operator applications in between never leave the device
// (PAPER.md:173 fn. c, 276) -- how the method uses an accelerator.  Uses the context's workspace.
extern "C" int lqcd_cg_multishift_host_vectors(lqcd_ctx *ctx, int nshift, const double *shifts, const void *rhs_host,
                                               void *solutions_host, const void *links_native_dev, double mass,
                                               double tol, int max_iter, int *iters, int *conv_iter, double *rel_resid)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return lqcd_fail(ctx, LQCD_ERR_ARG, "nshift %d not in [1,%d]", nshift, LQCD_MAX_SHIFTS);
    if (!rhs_host || !solutions_host || !links_native_dev || !shifts) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_cg_multishift_host_vectors: null pointer");
    const size_t canon_sp = (size_t)ctx->g.Vh * 3 * 16, csp = up256(canon_sp);
    const size_t nat_sp = up256(lqcd_spinor_bytes(ctx));
    if ((rc = stage_reserve(ctx, 2 * csp + (size_t)(1 + nshift) * nat_sp))) return rc;
    char *c_sp[2] = { (char *)ctx->stage, (char *)ctx->stage + csp };
    char *n_b = (char *)ctx->stage + 2 * csp, *n_x = n_b + nat_sp;
    cudaStream_t s = ctx->stream;
    if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync(c_sp[0], rhs_host, canon_sp, cudaMemcpyHostToDevice, s), "H2D rhs"))) return rc;
    if ((rc = lqcd_pack_spinor(ctx, LQCD_EVEN, n_b, c_sp[0]))) return rc;
    void *xs[LQCD_MAX_SHIFTS];
    for (int i = 0; i < nshift; ++i) xs[i] = n_x + (size_t)i * nat_sp;
    int solve_rc = lqcd_cg_multishift(ctx, nshift, shifts, n_b, xs, links_native_dev, mass, tol, max_iter, iters, conv_iter, rel_resid);
    if (solve_rc != LQCD_OK && solve_rc != LQCD_ERR_NOT_CONVERGED) return solve_rc;
    for (int i = 0; i < nshift; ++i) {     // (the stream orders unpack i+2 after the download of i from the same slot)
        if ((rc = lqcd_unpack_spinor(ctx, LQCD_EVEN, c_sp[i & 1], xs[i]))) return rc;
        if ((rc = lqcd_check_cuda(ctx, cudaMemcpyAsync((char *)solutions_host + (size_t)i * canon_sp, c_sp[i & 1], canon_sp, cudaMemcpyDeviceToHost, s), "D2H solution"))) return rc;
    }
    if ((rc = lqcd_check_cuda(ctx, cudaStreamSynchronize(s), "lqcd_cg_multishift_host_vectors"))) return rc;
    return solve_rc;
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
