/*
 * helios_rt_debug.h -- NOT part of the product API (include/helios_rt.h).  Launch-shape overrides of the RT step for
 * tests/ and for tuning runs: the library picks its launch shape from the problem sizes alone (never from the
 * environment); these two calls let a test force every compiled shape through the same parity checks.
 */
#ifndef HELIOS_RT_DEBUG_H
#define HELIOS_RT_DEBUG_H

#include "helios_rt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Re-selects the compiled instantiation of rt_step_kernel and the block size of a handle.  A value <= 0 (warps, ppt)
 * or < 0 (the others) keeps the current / any value.  warps: warps per block (1..maxt/32); ppt: spectral points per
 * thread (1, 2, 4; n_gauss must be a multiple; non-isothermal handles: 1 or 2); rows: 0 = k-table rows by
 * register-prefetched loads, 1 = by bulk async copies (TMA) into the per-warp shared-memory ring; maxt, minb: the launch
 * bounds the instantiation was compiled with (register cap = 65536 / (maxt * minb)).  HELIOS_RT_EINVAL if no such instantiation was
 * compiled or the shape does not fit an SM; the handle is then unchanged.  Re-allocates the shape-dependent workspace:
 * must not be called while a step of this handle is in flight. */
int helios_rt_debug_set_launch(helios_rt *h, int32_t warps, int32_t ppt, int32_t rows, int32_t maxt, int32_t minb);

/* Caps the number of workers (persistent blocks) per tile of the spectral axis; 0 removes the cap.  The default grid is
 * as many blocks as are resident at once (SMs x blocks per SM / tiles); fewer workers shrink the back-substitution
 * workspace (one slab per block of the grid) at the price of idle block slots -- a tuning knob for measuring that
 * trade, not something the product path sets.  Re-allocates the workspace like set_launch. */
int helios_rt_debug_set_workers(helios_rt *h, int32_t workers);

/* on != 0: every later step of the handle is launched WITHOUT its phase A, with a poll limit of 64: no column is ever
 * published, every block gives up waiting and the step must be reported as HELIOS_RT_ESTUCK (by helios_rt_step_host at
 * once, by the call after an asynchronous helios_rt_step).  Such a step sweeps whatever the workspace holds: call it
 * only after a normal step of the same handle on the same inputs (an uninitialised workspace holds wild table indices).
 * Lets a test see the error path that a healthy GPU never takes. */
int helios_rt_debug_force_stuck(helios_rt *h, int32_t on);

/* on != 0: every later step of the handle takes the path the library falls back to when the device cannot host the
 * whole grid of rt_step_kernel at once (cooperative launch refused): phase A as a launch of its own (rt_prep_kernel),
 * then the sweeps as a plain launch.  Lets the tests run that path through the parity checks. */
int helios_rt_debug_force_two_launches(helios_rt *h, int32_t on);

/* info[0] = warps per block, [1] = points per thread, [2] = rows, [3] = 0 (unused), [4] = maxt, [5] = minb, [6] = tiles per
 * column, [7] = workers per tile (grid = tiles x workers), [8] = resident blocks per SM, [9] = registers per thread,
 * [10] = local-memory bytes per thread, [11] = dynamic shared memory bytes, [12] = back-substitution workspace in MiB,
 * [13] = index of the instantiation, [14] = number of compiled instantiations, [15] = 0. */
int helios_rt_debug_get_launch(const helios_rt *h, int32_t info[16]);

#ifdef __cplusplus
}
#endif
#endif /* HELIOS_RT_DEBUG_H */
