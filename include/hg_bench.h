/* hg_bench.h -- measurement helpers of libhg.so for bench.py and the profiles.  NOT part of the product boundary
 * (include/hg.h): nothing here is a step of the path; a user of the library never needs these calls. */
#ifndef HG_BENCH_H
#define HG_BENCH_H

#include "hg.h"

#ifdef __cplusplus
extern "C" {
#endif

/* hg_set_profiling(ctx, 1) makes hg_integrate_step record CUDA events on the
 * launching stream around its kernels; hg_last_step_info then returns, for the last hg_integrate_step of the
 * context, out[0] = milliseconds spent in phase-space kernels (0 when the step is one fused kernel), out[1] =
 * milliseconds in the kernel(s) that evaluate the matrix element, out[2] = number of kernels launched. */
int hg_set_profiling(hg_ctx* ctx, int on);
int hg_last_step_info(const hg_ctx* ctx, double out[3]);

/* Measured-peak helper for the roofline: runs a register-resident FMA chain on every SM
 * and returns the achieved FLOP/s for the given precision in *flops_per_s.  Synchronises. */
int hg_measure_fma_peak(hg_ctx* ctx, int precision, double* flops_per_s, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* HG_BENCH_H */
