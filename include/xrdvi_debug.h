/*
 * xrdvi_debug.h -- read-back and measurement entry points of libxrdvi.so that are NOT part of the product boundary
 * (include/xrdvi.h): the parity tests read the draws and the forward pass back through them, bench.py and the
 * profiling runs time the kernels through them.  Same rules as xrdvi.h (return codes, host pointers unless stated,
 * no allocation inside the library: scratch memory is DEVICE memory owned by the caller).
 */
#ifndef XRDVI_DEBUG_H
#define XRDVI_DEBUG_H

#include "xrdvi.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Debug read-back of the forward pass for parity tests: runs draw + forward at (var_params or
 * internal state, S, seed, iteration) and returns, for the n sample-instances first .. first + n - 1 in
 * (pat, rst, s) order, the profile f float [n][N] (including B) and ll double [n]; f or ll may be NULL.
 * scratch: DEVICE buffer of at least n * N floats when f is wanted (XRDVI_E_WORKSPACE_TOO_SMALL otherwise). */
int xrdvi_debug_profile(xrdvi* h, const float* var_params, int32_t S, uint64_t seed,
                        uint64_t iteration, int64_t first, int64_t n, float* f, double* ll, void* scratch,
                        size_t scratch_bytes);

/* Debug read-back of the draw kernel (a-1, a-2) at the internal state: eps float [n][K][4] for the first n
 * sample-instances; raw_words uint32 [n][K][4] (the Philox output) or NULL; core_halfwidth int32 [n][K]
 * or NULL: the Gaussian-core half-width n_g in grid points of the 32-draw group the instance belongs to
 * (outside |i - j_m| <= n_g the kernels evaluate only the Lorentzian).
 * scratch: DEVICE buffer of at least 16 * P * R * ceil(S / 32) * 32 * K bytes.                           */
int xrdvi_debug_draws(xrdvi* h, int32_t S, uint64_t seed, uint64_t iteration, int64_t n, float* eps,
                      uint32_t* raw_words, int32_t* core_halfwidth, void* scratch, size_t scratch_bytes);

/* Measurement: mean CUDA-event times (ms) over `reps` repetitions (after one warm-up) of the kernels of one
 * evaluation at the internal state, launched one by one on the handle's stream: ms float [4] =
 * [0] elbo_tile_kernel (fused profile + residual + backward), [1] its forward-only instantiation (profile +
 * residual), [2] update_draw_kernel without the update, [3] draw + tile + update together.          */
int xrdvi_time_kernels(xrdvi* h, int32_t S, uint64_t seed, int32_t reps, float* ms);

/* Measurement: per-warp timeline of ONE launch of the fused profile / residual / backward kernel (a-3 .. a-7) at the
 * internal state with S draws per instance, after two un-stamped warm-up launches.  Every warp (or, where the
 * ticket-queue variant of the kernel is selected, every one-warp work item) writes four uint64 words:
 *   [0] %globaltimer (ns) when it starts, [1] at the end of the profile phase, [2] when it is done,
 *   [3] SM id (low 32 bits) | number of (peak, tile) records of its share (high 32 bits).
 * rows uint64 [capacity][4] (host), *n_rows = rows written; XRDVI_E_INVALID_ARG if capacity is smaller than the
 * number of warps of the launch; scratch: DEVICE buffer of 32 bytes per warp of the launch.  The state is not modified
 * (the per-step draw buffers are overwritten).                                                              */
int xrdvi_debug_timeline(xrdvi* h, int32_t S, uint64_t seed, int64_t capacity, uint64_t* rows, int64_t* n_rows,
                         void* scratch, size_t scratch_bytes);

/* Measurement: timeline of ONE launch of update_draw_kernel (a-6 prior part, a-7, a-8 and the next a-1 / a-2), the serial
 * section between two tile kernels.  Runs `steps` >= 2 optimisation steps from the internal state (the state advances) as
 * xrdvi_fit enqueues them (programmatic dependent launches, outside a graph); in the last step but one thread 0 of every CTA of
 * update_draw_kernel (an instantiation with the stamps compiled in; the product launches have none) writes eight
 * %globaltimer words (ns):
 *   [0] the CTA is resident, [1] it is done with everything that needs no output of the tile kernel (parameters, moments,
 *   prior terms, bias corrections, Philox normals of the next draws), [2] its griddepcontrol.wait returned, [3] the output
 *   slots (log-likelihood CTAs: the tiles) are added, [4] shuffle trees and barrier of the block reduction, [5] the
 *   parameter of thread 0 is updated, [6] all parameters of the phase are (0 for log-likelihood CTAs and evaluations),
 *   [7] the CTA is done.
 * Rows are CTAs in launch order (instance-major: K phase CTAs, then the log-likelihood CTAs of the instance); one more row
 * follows whose word [0] is the time at which the first warp of the NEXT step's tile kernel was past its
 * griddepcontrol.wait (the earliest start stamp of xrdvi_debug_timeline's rows, taken in the last step) and whose
 * word [1] is the time at which the last warp of the SAME step's tile kernel was done (its stamps slow that launch by
 * about 5 %, not the hand-over).
 * rows uint64 [capacity][8] (host), *n_rows = CTAs + 1; XRDVI_E_INVALID_ARG if capacity is smaller; scratch: DEVICE
 * buffer of 64 bytes per CTA of update_draw_kernel + 64 bytes per warp of the tile kernel's launch.              */
int xrdvi_debug_update_timeline(xrdvi* h, int32_t steps, int32_t S, uint64_t seed, int64_t capacity, uint64_t* rows,
                                int64_t* n_rows, void* scratch, size_t scratch_bytes);

/* Measurement: `steps` optimisation steps (graph replays, exactly as xrdvi_fit runs them), each one
 * bracketed by its own pair of CUDA events on the handle's stream; between two steps, outside the
 * brackets, the DEVICE buffer l2_flush (l2_flush_bytes; NULL / 0 = no flush) is overwritten so that every step
 * starts with a cold L2.  ms_steps float [steps] receives the per-step device times.  The state advances.   */
int xrdvi_bench_steps(xrdvi* h, int32_t steps, int32_t S, uint64_t seed, void* l2_flush, size_t l2_flush_bytes,
                      float* ms_steps);

#ifdef __cplusplus
}
#endif
#endif /* XRDVI_DEBUG_H */
