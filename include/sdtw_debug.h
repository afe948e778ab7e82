/*
 * sdtw_debug.h -- instrumentation and tuning hooks of libsdtw.  NOT part of the numerical path and not part of the
 * product boundary (include/sdtw.h): bench.py and the tests use them to time kernels, to measure the roofline
 * denominator and to prove that scheduling / skipping choices do not change a result bit.
 *
 * All switches below (profiling on/off, reverse mode, forward schedule) are PER CALLING THREAD: they affect only the
 * library calls the same host thread makes afterwards, so one thread's measurement settings never change another
 * thread's launch.
 */
#ifndef SDTW_DEBUG_H_
#define SDTW_DEBUG_H_

#include "sdtw.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Instrumentation used by bench.py (not part of the numerical path).
 *   sdtw_launch_count()   kernels launched by this library since load.
 *   sdtw_profile_enable() when on, every sdtw_value_grad / barycenter iteration brackets its forward kernel, its
 *                         reverse kernel and the remaining small kernels with CUDA events on the caller's stream.
 *   sdtw_profile_read()   waits for those events and returns the accumulated milliseconds and the number of
 *                         evaluations they cover; clears the accumulators.  Any pointer may be NULL.
 */
uint64_t sdtw_launch_count(void);
/* Waves of pairs (sdtw.h, "WAVES") the calling thread's last sdtw_value_grad[_ex] / sdtw_barycenter[_ex] / DTW call was
 * evaluated in: 1 = unsplit, 0 = no such call yet.  A call that splits does so silently (same values); a caller that
 * shares the GPU with a caching allocator can watch this number to notice that its budget has become small. */
int sdtw_last_wave_count(void);
int sdtw_profile_enable(int on);
int sdtw_profile_read(double* ms_forward, double* ms_backward, double* ms_other, int64_t* evaluations);

/*
 * sdtw_measure_mufu_peak -- measurement, not part of the numerical path: runs dependent chains of one special-function
 * instruction (kind 0 = ex2.approx, 1 = lg2.approx, 2 = rcp.approx; the three the kernels use) on every SM of the
 * current device on a private stream, BLOCKS until done, and returns results per second (best of 3) and the SM count.
 * This is the denominator of the roofline bench.py reports.
 */
int sdtw_measure_mufu_peak(int32_t kind, double* ops_per_s, int32_t* sm_count);

/*
 * Reverse-pass mode.  The expected-alignment matrix E of eq. 6 underflows to exactly +0 in float32 away from the
 * alignment band, and every quantity the reverse recurrence derives from zero flows is +0 as well; by default the
 * reverse kernel therefore SKIPS a 32-step chunk of a column strip when every flow entering it is +0.  The result is
 * bitwise identical to visiting every cell.  sdtw_set_reverse_mode(1) disables the skip (every cell is visited: the
 * "dense" mode used for measurement and for the bitwise-equality test); 0 restores the default.
 * sdtw_reverse_stats() BLOCKS (device synchronise) and returns, for the last evaluation that ran a reverse pass, the
 * number of (strip, chunk) units and how many of them were skipped.  Either pointer may be NULL.
 */
int sdtw_set_reverse_mode(int dense);
int sdtw_reverse_stats(uint64_t* chunks, uint64_t* skipped);
/*
 * The reverse pass has two kernels with the same arithmetic: 1 = reverse_kernel (a CTA of four warps per
 * column strip; the recompute runs off the pair's dependency chain: the latency regime), 0 = backward_kernel (one warp
 * per strip, four times as many strips in flight: the throughput regime, and the dense mode).  -1 (default) chooses by
 * the number of pairs and the reverse mode.  Results agree to float32 round-off of the per-column sums (the order in
 * which a column's rows are added differs); each kernel is bitwise reproducible.  Other values => SDTW_ERR_INVALID_ARG.
 */
int sdtw_set_reverse_kernel(int which);
/*
 * Forward-only calls without a band (and the DTW calls at d <= 2) can pass strip-boundary values through per-warp
 * rings inside a unit of strips instead of keeping one boundary column per strip (sdtw_kernels.cuh).  1 (default): when
 * the problem has more strips than resident warps AND the columns would take more than 6 GB (1000 cycles of 30k: 28 GB
 * of columns, 1 GB with rings, 1 % slower; a few hundred cycles are faster with columns, whose schedule can end with
 * small units).  2: whenever the problem has more strips than resident warps.  0: never (the workspace then has to be
 * sized with sdtw_workspace_bytes_ex and a band that excludes a cell).  The values are bitwise the same.
 * Other values => SDTW_ERR_INVALID_ARG.
 */
int sdtw_set_forward_rings(int on);

/*
 * Forward schedule (tuning, does not change any result bit): the forward kernel hands out UNITS of `unit_strips`
 * adjacent column strips of one pair to its CTAs (sdtw_kernels.cuh).  0 restores the automatic choice; values above
 * the kernel's warps per CTA are clamped.  Negative => SDTW_ERR_INVALID_ARG.
 */
int sdtw_set_schedule(int unit_strips);
/* The last `tail_strips` strips of every pair are handed out in units of `tail_unit` strips (small units at the end of
 * the queue shorten the drain).  tail_strips < 0 restores the automatic choice; tail_unit <= 0 means "as unit_strips". */
int sdtw_set_schedule_tail(int tail_strips, int tail_unit);

/* Compile-time tile constants, for DESIGN.md / bench.py reporting: columns per thread, columns per strip (work item),
 * wavefront steps between checkpoints, steps per strip-boundary exchange, rows a lane works on per step.  Any pointer
 * may be NULL. */
int sdtw_tile_info(int32_t* cols_per_thread, int32_t* strip_cols, int32_t* ckpt_steps, int32_t* chunk_steps,
                   int32_t* rows_per_step);

#ifdef __cplusplus
}
#endif
#endif /* SDTW_DEBUG_H_ */
