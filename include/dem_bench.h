/*
 * dem_bench.h -- measurement hooks of libdem_b200 (C ABI).  NOT part of the method: include/dem.h is the paper's problem
 * statement; these calls exist for bench.py, the profiling runs under profiles/ and the tests that check the counters.
 * Same conventions as dem.h (status codes, HOST / DEVICE pointers, the context's stream).
 */
#ifndef DEM_B200_BENCH_H
#define DEM_B200_BENCH_H

#include "dem.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Benchmark hygiene: when bytes > 0, dem_step overwrites a scratch buffer of that size (larger than the 126 MB L2)
 * before every time step, so that no step finds its inputs cached by the previous one.  0 (default) = off. */
int dem_set_l2_flush(dem_ctx* ctx, int64_t bytes);

/* Kernel-time accounting: CUDA events on the context's stream around the library's kernels.  level 0 = off (default);
 * 1 = the pose kernel and the pair-feature kernel of every evaluation; 2 = also the reduction, the integrator kernel,
 * the L2 flush and the neighbour build (k_neigh alone, and the whole build).  dem_kernel_times returns, per kernel
 * kind, the number of bracketed launches and their summed duration in milliseconds since the last call, and resets
 * them (synchronises).  A system with several pair classes (several shapes) runs its classes' pose and pair kernels on
 * side streams at the same time: it then reports ONE DEM_KT_PAIR span per evaluation, from the fork to the join (all pose
 * and pair kernels of the evaluation), and no DEM_KT_POSE spans. */
enum { DEM_KT_POSE = 0, DEM_KT_PAIR = 1, DEM_KT_REDUCE = 2, DEM_KT_KICK_DRIFT = 3, DEM_KT_NEIGH = 4, DEM_KT_BUILD = 5,
       DEM_KT_FLUSH = 6, DEM_KT_OTHER = 7, DEM_KT_COUNT = 8 };
int dem_set_timing(dem_ctx* ctx, int level);
int dem_kernel_times(dem_ctx* ctx, int64_t launches[DEM_KT_COUNT], double ms[DEM_KT_COUNT]);

/* While timing is on, the search kernels' swept-term counters (dem_get_counters out[7], out[6] - out[7], out[8]) are
 * also summed over all evaluations since dem_set_timing: out[0] edge-edge terms (2D: vertex-edge terms), out[1]
 * vertex-face terms, out[2] face boundary-edge tests.  HOST int64[3]; synchronises. */
int dem_swept_totals(dem_ctx* ctx, int64_t out[3]);

/* Number of kernels the library has launched on this context since creation (all kernels). */
int64_t dem_launch_count(const dem_ctx* ctx);

/* FP32 FMA-chain microbenchmark (roofline denominator): runs `iters` dependent-chain FFMA iterations on
 * every SM and returns the achieved FP32 TFLOP/s (2 flop per FMA); synchronises. */
int dem_fp32_peak(dem_ctx* ctx, int iters, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* DEM_B200_BENCH_H */
