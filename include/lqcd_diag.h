/*
 * lqcd_diag.h -- validation and measurement helpers exported by liblqcd_b200.so that are NOT part of the C ABI of
 * SURVEY.md section 8(b) (include/lqcd.h).  The tests, bench.py and sweep.py use them; an application has no reason to.
 * They may change or disappear without notice.  Also diagnostic, through lqcd_set_option: "iter_mask" (bit k set = kernel
 * k of the CG iteration is launched; results are INVALID unless 15, the default -- timing experiments only).
 */
#ifndef LQCD_DIAG_H
#define LQCD_DIAG_H

#include "lqcd.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Lock-step validation of the peer transport on ONE GPU.  The kernels of different ranks wait for one another, which must
 * never happen between launches on one device; lqcd_set_phase_hook installs a host callback that the library calls after
 * every launch that publishes to the peers (what = 0: face push, 1: generic all-reduce, 2: dot product).  A test harness
 * that synchronises its stream there and then meets the other ranks at a host barrier runs the ranks in lock step, so
 * that no kernel ever waits (the chunk graph is off while a hook is set).  Pass NULL to clear.
 */
typedef int (*lqcd_phase_fn)(void *user, int what);
int lqcd_set_phase_hook(lqcd_ctx *ctx, lqcd_phase_fn fn, void *user);

/* Protocol self-test under real concurrency on ONE GPU: one cooperative kernel whose CTA r plays rank r of `nranks` on its
 * own block -- the flags, slots and counters of the transport with ranks that really run at the same time, at uneven pace,
 * and really wait for one another -- for `rounds` iterations of (halo exchange, two all-reduces).  *failures = wrong
 * tokens / sums / waits that gave up (0 = pass).  sabotage = 1 makes the consumers skip their waits: the count must then
 * be non-zero for more than a few ranks (the check that the test can fail).  Allocates and frees its own scratch memory;
 * independent of lqcd_peer_init.  blocking. */
int lqcd_peer_selftest(lqcd_ctx *ctx, int nranks, int rounds, int sabotage, int *failures);

/*
 * Measurement helper (no arithmetic of the method): attainable FP64 FMA rate of the device in TFLOP/s, from a
 * kernel of independent DFMA chains on the context's stream -- the roofline denominator of the ALU-bound
 * gauge-staples kernel (bench.py extra.fp64_peak_tflops).  tflops: host, out.  blocking.
 */
int lqcd_measure_fp64_peak(lqcd_ctx *ctx, double *tflops);
/* Measurement helper: attainable READ bandwidth in GB/s over the caller's device buffer (use one larger than L2, e.g.
 * the link field): 16-byte streaming loads, nothing written.  MEASURED_PEAKS.json's HBM figure is a copy (half
 * writes); the Dslash is 96 % reads (bench.py roofline.frac_of_read_rate).  buf: 16-byte aligned, >= 1 MiB.  blocking. */
int lqcd_measure_hbm_read(lqcd_ctx *ctx, const void *buf_dev, size_t bytes, double *gbs);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_DIAG_H */
