/*
 * numa_b200_measure.h -- MEASUREMENT entry points of libnuma_b200.so (bench.py only).
 *
 * Kept apart from the product ABI (numa_b200.h): nothing here is needed to run the hot path
 * of arXiv 2504.08157 (Eq. 1-12, Alg. 1-3); these calls only time it, count its
 * launches and measure the FP64 ceiling it is compared with ("whichever of
 * HBM or FP64 binds"; BASELINE.json north_star: "FP64 FLOP/s against peak").
 */
#ifndef NUMA_B200_MEASURE_H
#define NUMA_B200_MEASURE_H

#include "numa_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Optional per-kernel timing with CUDA events recorded on the launching stream around every
 * kernel this context launches.  numa_profile_enable(ctx, 1) clears the accumulators and
 * starts recording, (ctx, 0) stops.  Off by default; bench.py times its headline with it off
 * and collects the per-kernel split in a second pass.  numa_profile_read waits for the
 * recorded events and returns the accumulated device time and launch count of one kernel id
 * (0 .. numa_kernel_count()-1); numa_kernel_name gives the kernel's name.
 * While profiling is on numa_step_rk3_graph uses plain launches.
 */
numa_status numa_profile_enable(numa_ctx *ctx, int32_t enable);
numa_status numa_profile_read(numa_ctx *ctx, int32_t kernel_id, double *total_ms, int64_t *launches);
const char *numa_kernel_name(int32_t kernel_id);
int32_t numa_kernel_count(void);

/* Number of kernel launches this context has enqueued so far (bench.py's gpu_launches);
 * a kernel replayed from a CUDA graph counts as one launch per replay. */
int64_t numa_launch_count(const numa_ctx *ctx);

/*
 * FP64 ceiling of the current device: a register-resident kernel of dependent-chain-free
 * DFMA (8 independent accumulators per thread, 1024 FMAs per accumulator per pass, grid =
 * SMs x resident blocks) timed with CUDA events on `stream`; *tflops = 2 * FMAs / time, best
 * of `repeats` launches after one warm-up.  This is the denominator of bench.py's FP64
 * roofline leg.  Synchronises `stream`.
 */
numa_status numa_measure_fp64_peak(int32_t repeats, double *tflops, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* NUMA_B200_MEASURE_H */
