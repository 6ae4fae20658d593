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

#ifdef __cplusplus
}
#endif
#endif
