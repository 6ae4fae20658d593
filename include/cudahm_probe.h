/*
 * cudahm_probe.h -- measurement probes exported next to the sampler (same library).
 *
 * BASELINE.json north_star asks that "per-iteration launch and sync cost is measured" and that the fp64/fp32
 * pipe peak be the secondary roofline; MEASURED_PEAKS.json has neither, so the library measures them with the
 * very mechanisms the sampler uses.  All times are CUDA-event times on `stream`.
 */
#ifndef CUDAHM_PROBE_H
#define CUDAHM_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif

enum { CUDAHM_FLOOR_LAUNCH = 0,      /* n back-to-back launches of an empty kernel pair (sweep-sized + 1 warp)   */
       CUDAHM_FLOOR_GRAPH = 1,       /* the same pair captured 50x in a CUDA graph, replayed                     */
       CUDAHM_FLOOR_GRID_BARRIER = 2,/* one cooperative launch looping n times over the sampler's grid barrier    */
       CUDAHM_FLOOR_HOST_SYNC = 3 }; /* launch + 40-byte D2H copy + stream sync per iteration (the paper's split) */

/* Per-iteration floor in microseconds for `kind`, with `grid_blocks` x `block_threads` (0 = one block per SM x 512).
 * Returns 0 or a negative CUDAHM_E_* code. */
int cudahm_probe_floor(void* cuda_stream, int kind, int n_iter, int grid_blocks, int block_threads, double* us_per_iter);

/* Register-resident FMA throughput of the plain ALU pipes, in tera-FMA/s: dtype 0 = fp64 (DFMA), 1 = fp32 (FFMA). */
int cudahm_probe_fma_peak(void* cuda_stream, int dtype, double* tera_fma_per_s);

/* The device builds of the elementary functions of csrc/fastmath.cuh, evaluated on the GPU: y[i] = fn(x[i]) for n HOST
 * doubles (copied in and out on `stream`, which is synchronised before the call returns).  The sampler's kernels call these
 * very functions; tests/test_gpu_fastmath.py holds their device results to the bounds the host builds are pinned to
 * (the device seeds its reciprocal and reciprocal square root with MUFU instructions the host cannot reproduce).
 * CUDAHM_MATH_SIN2PI / COS2PI: hm_sincos2pi (the Box-Muller angle, x in [0, 1]); SQRT_BOTH_*: the two results of
 * hm_sqrt_rsqrt.  Returns 0 or a negative CUDAHM_E_* code. */
enum { CUDAHM_MATH_EXP = 0, CUDAHM_MATH_EXPM1_NONPOS = 1, CUDAHM_MATH_LOG = 2, CUDAHM_MATH_SQRT = 3, CUDAHM_MATH_SQRT_BOTH_ROOT = 4,
       CUDAHM_MATH_SQRT_BOTH_INV = 5, CUDAHM_MATH_SIN2PI = 6, CUDAHM_MATH_COS2PI = 7,
       /* LOG .. SQRT_BOTH_INV above are the one-Newton-step variants; these are the two-step ones (fastmath.cuh, HM_NEWTON_STEPS) */
       CUDAHM_MATH_LOG_2 = 8, CUDAHM_MATH_SQRT_2 = 9, CUDAHM_MATH_SQRT_BOTH_ROOT_2 = 10, CUDAHM_MATH_SQRT_BOTH_INV_2 = 11 };
int cudahm_probe_math(void* cuda_stream, int fn, const double* x_host, double* y_host, long long n);

#ifdef __cplusplus
}
#endif
#endif
