/* etac_bench.h -- measurement entry points of libetac.so used by bench.py.  NOT part of the product ABI of
 * etac.h: nothing on the hot path calls them, and an application never needs them.  They live in the same
 * shared library because the per-kernel split of a step can only be timed from inside it (CUDA events between
 * the kernels of one etac_step on the launching stream). */
#ifndef ETAC_BENCH_H_
#define ETAC_BENCH_H_

#include "etac.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Timing helper for bench.py: times `iters` back-to-back etac_step calls on cuda_stream with CUDA
 * events recorded on that stream and returns the mean milliseconds per step in *ms_per_step
 * (host pointer).  If ms_kernels (host, [2]) is not NULL a second pass of `iters` steps records
 * events between the kernels: ms_kernels[0] = S1 (sdf_penetration, incl. its two small memsets),
 * ms_kernels[1] = fused S2+S3+S4 kernel, mean ms per launch.  Synchronises the stream on both sides. */
etac_status etac_time_steps(etac_ctx* ctx, void* cuda_stream, const etac_step_args* args, int32_t iters,
                            float* ms_per_step, float* ms_kernels);

/* Measurement helper for bench.py's roofline (not on the hot path): runs a microbenchmark of independent
 * tanh.approx.f32 chains on every SM of the current device, on cuda_stream, and returns the measured rate of
 * the special-function pipe in results per second (*ops_per_s, host pointer) and, if not NULL, per clock and
 * SM at the device's nominal maximum clock (*ops_per_clk_per_sm).  The fused kernel evaluates 128 SiLUs
 * (one MUFU.TANH each) per node-environment of a contacting pair, BASELINE.json configs[0] "2x64 SiLU"; this
 * rate is the denominator of its "alu" roofline.  Synchronises the stream.
 * Errors: ETAC_ERR_INVALID_ARG (NULL ops_per_s), ETAC_ERR_CUDA. */
etac_status etac_measure_sfu_rate(void* cuda_stream, double* ops_per_s, double* ops_per_clk_per_sm);

#ifdef __cplusplus
}
#endif
#endif /* ETAC_BENCH_H_ */
