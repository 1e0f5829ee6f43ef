// diag.cu -- measurement helpers of the C ABI (no arithmetic of the method).
// lqcd_measure_fp64_peak: the device's attainable FP64 FMA rate, the denominator of the roofline of the
// one ALU-bound kernel of the library (the gauge staples, staples.cu).  MEASURED_PEAKS.json
// holds HBM and bf16 figures only, so bench.py measures this one itself, in the same process and under the
// same clocks as the kernel it is compared with.
#include "common.cuh"

// 16 independent DFMA chains per thread (enough to cover the FP64 pipe's latency at 8+ warps per scheduler),
// 8 CTAs of 256 threads per SM: nothing but dependent-free FMAs in the loop.
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *sink, int iters, double a, double b)
{
    double x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = (double)(threadIdx.x + k) * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) x[k] = fma(x[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    if (s == 123.456) sink[0] = s;      // never true: keeps the chains alive without a store per thread
}

extern "C" int lqcd_measure_fp64_peak(lqcd_ctx *ctx, double *tflops)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!tflops) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_measure_fp64_peak: null pointer");
    const int iters = 1 << 13, grid = ctx->num_sms * 8, block = 256;
    cudaEvent_t e0, e1;
    if ((rc = lqcd_check_cuda(ctx, cudaEventCreate(&e0), "event"))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaEventCreate(&e1), "event"))) { cudaEventDestroy(e0); return rc; }
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {      // first repetitions warm the clocks up; best of the rest
        cudaEventRecord(e0, ctx->stream);
        fp64_peak_kernel<<<grid, block, 0, ctx->stream>>>((double *)ctx->d_partials, iters, 0.999999, 1e-9);
        ctx->launches++;
        cudaEventRecord(e1, ctx->stream);
        cudaError_t e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return lqcd_check_cuda(ctx, e, "fp64 peak kernel"); }
        const double flop = 2.0 * 16.0 * (double)iters * (double)grid * (double)block;
        const double tf = flop / ((double)ms * 1e-3) / 1e12;
        if (rep >= 2 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops = best;
    return LQCD_OK;
}

// lqcd_measure_hbm_read: the device's attainable READ bandwidth over a caller buffer larger than L2 (16-byte
// streaming loads, one resident wave looping, a sum that is never stored).  MEASURED_PEAKS.json's figure is a COPY
// (half writes); the Dslash is 96 % reads and reads run faster than a copy on HBM3e, which is why its fraction of the
// copy peak exceeds 1 -- bench.py reports the fraction of this read rate beside it.
__global__ void __launch_bounds__(256) hbm_read_kernel(const double2 *__restrict__ p, size_t n, double *sink)
{
    // 8 independent 16-byte loads in flight per thread (one per trip left the kernel latency-bound below the Dslash's
    // own rate)
    double s = 0.0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t k = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    for (; k + 7 * stride < n; k += 8 * stride) {
        double2 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = __ldcs(p + k + u * stride);
#pragma unroll
        for (int u = 0; u < 8; ++u) s += v[u].x + v[u].y;
    }
    for (; k < n; k += stride) {
        const double2 v = __ldcs(p + k);
        s += v.x + v.y;
    }
    if (s == 123.456) sink[0] = s;      // practically never: keeps the loads alive
}

extern "C" int lqcd_measure_hbm_read(lqcd_ctx *ctx, const void *buf, size_t bytes, double *gbs)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!buf || !gbs || ((uintptr_t)buf & 15) || bytes < (size_t)1 << 20)
        return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_measure_hbm_read: null / unaligned pointer or fewer than 1 MiB");
    const size_t n = bytes / 16;
    const int grid = ctx->num_sms * 8, block = 256;
    cudaEvent_t e0, e1;
    if ((rc = lqcd_check_cuda(ctx, cudaEventCreate(&e0), "event"))) return rc;
    if ((rc = lqcd_check_cuda(ctx, cudaEventCreate(&e1), "event"))) { cudaEventDestroy(e0); return rc; }
    double best = 0.0;
    for (int rep = 0; rep < 8; ++rep) {
        cudaEventRecord(e0, ctx->stream);
        hbm_read_kernel<<<grid, block, 0, ctx->stream>>>((const double2 *)buf, n, (double *)ctx->d_partials);
        ctx->launches++;
        cudaEventRecord(e1, ctx->stream);
        cudaError_t e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return lqcd_check_cuda(ctx, e, "hbm read kernel"); }
        const double g = (double)(n * 16) / ((double)ms * 1e-3) / 1e9;
        if (rep >= 2 && g > best) best = g;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *gbs = best;
    return LQCD_OK;
}
