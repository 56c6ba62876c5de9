/* paraiso_hydro.h — C ABI of the B200-native Euler hot path (libparaiso_hydro.so).
 *
 * What the library computes: explicit time steps of the finite-volume compressible Euler solver
 * that Paraiso generates (arXiv 1204.4779 §4.1) on a uniform Cartesian grid in
 * 1, 2 or 3 dimensions, plus the global CFL reduction that sets dt:
 *   Eq. 19 primitive recovery, Eq. 20-21 MINBEE reconstruction, Eq. 22 HLLC (or HLL) flux,
 *   Eq. 23 flux-divergence update, Eq. 24-27 two-stage (midpoint) Runge-Kutta.
 * Readings of the paper and the written arithmetic: DESIGN.md §3-4.
 *
 * Conventions
 *   - State = CONSERVED variables U = (rho, m_x[, m_y[, m_z]], E) (Eq. 14), nf = dims+2
 *     fields, SoA, field-major, x fastest:  U[f*N + (k*n[1] + j)*n[0] + i],  N = prod n[a].
 *     Element type float (PARAISO_F32) or double (PARAISO_F64), fixed at create.
 *   - Pointers named "host or device" may be either; the library asks cudaPointerGetAttributes.
 *     Device pointers must belong to the current device. Managed memory counts as device.
 *   - Ownership: the caller owns every pointer it passes in; the handle owns all internal device
 *     buffers. set_state / get_state copy.
 *   - Every function returns PARAISO_OK (0) or a negative error code; no exception crosses the ABI;
 *     paraiso_hydro_last_error() returns a static or per-handle message for the last failure.
 *   - All work is enqueued on the handle's stream (default: the legacy default stream; see
 *     set_stream). Blocking calls: cfl_dt, get_state to host memory, run (only when t_end > 0),
 *     sync, stats, time. step() is asynchronous.
 *   - There is no CPU fallback: create() fails with PARAISO_ECUDA when no CUDA device is usable.
 *   - A handle is not thread-safe; distinct handles are independent.
 */
#ifndef PARAISO_HYDRO_H
#define PARAISO_HYDRO_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct paraiso_hydro paraiso_hydro_t;

enum { PARAISO_F32 = 0, PARAISO_F64 = 1 };

enum {
  PARAISO_OK = 0,
  PARAISO_EINVAL = -1,     /* bad argument (null pointer, dims, sizes, gamma, dt, unknown option) */
  PARAISO_ENOMEM = -2,     /* device allocation failed */
  PARAISO_ECUDA = -3,      /* CUDA runtime error or no device */
  PARAISO_ESTATE = -4,     /* step / cfl_dt / get_state / run before set_state */
  PARAISO_ENONFINITE = -5  /* reported by stats(): non-finite or non-positive rho / p was seen */
};

/* Create a solver for a dims-dimensional periodic box (dims = 1, 2, 3).
 *   n[dims]      cells per axis, x first; every n[a] >= 4 (the stencil of one stage reaches 2 cells)
 *   extent[dims] physical edge lengths; mesh size dr_a = extent[a] / n[a]  (Eq. 23 "Delta r_a")
 *   gamma        ratio of specific heats of the ideal-gas EOS E = p/(gamma-1) + rho v^2/2, > 1
 *   dtype        PARAISO_F32 | PARAISO_F64 — the arithmetic type of the whole path
 * Size limit: N = prod n[a] <= 2^31 / 8 = 268 435 456 cells (645^3; 16384^2), because every kernel addresses the
 * nf * N elements of a state buffer with 32-bit element offsets (index arithmetic is part of the issue-bound hot loop);
 * a larger grid is EINVAL, not a wrong answer.  The five BASELINE configs need at most 512^3 = 2^27.
 * Allocates two state buffers (2 * nf * N elements) and a small scalar block on the current device.
 * Errors: EINVAL, ENOMEM, ECUDA.  *out is set only on success. */
int paraiso_hydro_create(paraiso_hydro_t **out, int dims, const int64_t *n, const double *extent, double gamma,
                         int dtype);

/* Release every device buffer and the handle.  NULL is accepted. */
int paraiso_hydro_destroy(paraiso_hydro_t *h);

/* Options (set before set_state or between steps).  Unknown key or value -> EINVAL.
 *   "boundary"  0 periodic: index wrap (default) | 1 outflow: zero-gradient, index clamp   (R12)
 *   "riemann"   0 HLLC (default; Eq. 22) | 1 HLL                              (R4)
 *   "variant"   kernel arrangement on the paper's Manifest <-> Delayed axis (Table 5):
 *               0 fused       one kernel per RK stage, intermediates on chip (default): k_pack on 2-D and 3-D grids
 *                             (fp32: packed pairs of cells, needs an even n_x, else k_march; fp64: one cell per
 *                             thread); in 1-D k_small1d up to 1024 cells (any number of steps in ONE launch, the
 *                             state in registers), k_delayed beyond
 *               6 pack        force k_pack (marching window in shared memory; the fastest on-chip kernel)
 *               4 march       force k_march (marching window in registers; "cells_per_thread" 2 = packed f32x2)
 *               5 fused1      force k_fused (the first on-chip design)
 *               1 manifest_flux  fluxes F_a materialised in HBM, then an update kernel
 *               2 manifest_all   V, VL/VR and F_a all materialised in HBM, one kernel per piece
 *               3 delayed     one kernel per stage, every thread recomputes all it needs from U
 *               An explicitly requested kernel, or any launch-shape knob, that does not cover the grid makes the next
 *               step / run return EINVAL ("shape not covered"); only variant 0 with all-default knobs falls back
 *               (pack -> march -> fused1 -> delayed).  get_option("kernel_used") = the kernel of the last stage launch.
 *   "block_x" "block_y" "block_z" "tile_depth" "cells_per_thread"   launch-shape knobs of the sweep (0 = default):
 *               k_pack: block_x = warps per row (2-D: 2, 4, 8 [fp32 also 1] as overlapping tiles without a halo warp;
 *               with block_z = 1 the halo-warp form, 2, 4, 7), block_y = tile rows (3-D: 7 [default on small grids],
 *               14 [two halo warps, default on large grids]; fp32 also 5, 11, 15); k_fused: block_x x block_y = tile;
 *               k_march: block_x = main warps per row (2-D), block_y = main warps (3-D), block_z = rows per main
 *               thread (3-D: 1 or 2), cells_per_thread 2 = packed f32x2; tile_depth = planes marched per block
 *               (0: chosen from the kernel's occupancy so that the grid fills whole waves).  A knob the selected
 *               kernel does not read in this dimension (k_pack / k_march: block_y in 2-D, block_x in 3-D, ...) must be
 *               0, and staging / arith are honoured in the default tile of k_march only: anything else is EINVAL
 *   "limiter"   interpolation variant (R22): 0 the paper's MINBEE, Eq. 21 (default) | 1 none: piecewise
 *               constant states, the first-order Godunov scheme | 2 monotonized central (van Leer 1977).  1 and 2 are
 *               compile-time variants of k_pack (default launch shape only) and k_delayed; any other kernel -> EINVAL
 *   "graph"     1 replay steps of run() from a captured CUDA graph (default) | 0 plain launches
 *   "arith"     k_march, fp32 only: 0 IEEE-exact division and square root, bit-equal to the oracle (default) |
 *               1 hardware reciprocal / reciprocal-square-root approximations: inside north_star's fp32 tolerances,
 *               not bit-equal, ~15 % faster (R21)
 *   "staging"   k_march only: 0 / 1 every thread loads its own cells (default) | 2 TMA bulk copies of the tile rows into a
 *               shared-memory ring (cp.async.bulk; one cell per thread, n_x a multiple of 16 bytes, else EINVAL) | 3 the same ring
 *               filled by one tensor-map copy per plane (cp.async.bulk.tensor); both measured, DESIGN.md §7
 *   "integrator" 0 the paper's two-stage midpoint rule, Eq. 24-27 (default) | 1 Heun / Shu-Osher SSP-RK2, the
 *               "2-stage TVD Runge-Kutta" north_star names as the fallback (R20): same kernels and traffic
 *   "state_kind" 0 set_state / get_state exchange conserved variables U = (rho, m_a, E) (default) |
 *               1 primitive variables V = (rho, v_a, p): converted on the device with the EOS of PAPER.md:694
 *               (set_state) and by Eq. 19 (get_state); the state inside the handle is always conserved */
int paraiso_hydro_set_option(paraiso_hydro_t *h, const char *key, int64_t value);
int paraiso_hydro_get_option(paraiso_hydro_t *h, const char *key, int64_t *value);

/* Use `cuda_stream` (a cudaStream_t, e.g. torch.cuda.Stream().cuda_stream; NULL/0 = legacy default)
 * for all subsequent work.  The caller keeps the stream alive. */
int paraiso_hydro_set_stream(paraiso_hydro_t *h, void *cuda_stream);

/* Copy nf*N elements of conserved variables from U (host or device) into the handle, reset t = 0 and
 * the step counter, and enqueue the standalone CFL reduction for this state.  The copy is asynchronous on the
 * handle's stream when U is a device pointer or pinned host memory: the caller keeps U alive (and unchanged) until the
 * stream has passed it (paraiso_hydro_sync, or any blocking call of this handle). */
int paraiso_hydro_set_state(paraiso_hydro_t *h, const void *U);

/* Copy the current state (nf*N elements) to U_out (host or device).  Host destination: blocks until done. */
int paraiso_hydro_get_state(paraiso_hydro_t *h, void *U_out);

/* dt = Real(cfl) / S,  S = max over cells and axes of (|v_a| + c) / dr_a of the CURRENT state, c = sqrt(gamma p / rho)
 * (R6).  After set_state S comes from the standalone reduction; after a step it was already produced by
 * the fused epilogue of that step's last stage, so this call only reads one scalar.  Blocking.  cfl > 0. */
int paraiso_hydro_cfl_dt(paraiso_hydro_t *h, double cfl, double *dt_out);

/* One full RK2 step (Eq. 24-27) with the given dt (rounded to the handle dtype; finite, > 0): t += dt.
 * Asynchronous.  The last stage also leaves S of the new state on the device. */
int paraiso_hydro_step(paraiso_hydro_t *h, double dt);

/* Prescribed ghost cells (the paper's validation runs "substitute the analytic solutions to the ghost cells",
 * PAPER.md:846-848; R23).  In this use the outermost TWO cells of every axis of the grid are the ghost cells
 * (two = the reach of the stencil of Eq. 20-22): the caller overwrites them with its own values, the cells in between
 * are advanced by Eq. 23-27 as always; "boundary" should be 1 (clamp), what the scheme computes in the ghost cells
 * themselves is overwritten before anything reads it.  G, G_mid: nf*N elements laid out like the state (host or
 * device; same lifetime rule as set_state), of which only the ghost cells are read.
 *   set_ghosts   ghost cells of the CURRENT state := G's (call it before every step with the ghosts of time t, and
 *                after the last step if the ghost cells of the result matter); it does not refresh S: pass your own dt
 *   step_ghosts  one RK2 step like paraiso_hydro_step, but the ghost cells of the intermediate state U1 := G_mid's
 *                before the second stage (midpoint rule: the ghosts of time t + dt/2; Heun: of time t + dt) */
int paraiso_hydro_set_ghosts(paraiso_hydro_t *h, const void *G);
int paraiso_hydro_step_ghosts(paraiso_hydro_t *h, double dt, const void *G_mid);

/* Advance with dt from the CFL condition evaluated on the device at the start of every step, without host
 * round trips: at most nsteps steps; if t_end > 0 stop when t reaches t_end, the last step clamped to land on it
 * exactly (R18).  With t_end <= 0 the call only enqueues work (asynchronous) and *steps_done = nsteps,
 * *t_out is not written; with t_end > 0 it blocks and reports the steps taken and the final time.
 * steps_done, t_out may be NULL. */
int paraiso_hydro_run(paraiso_hydro_t *h, double cfl, int64_t nsteps, double t_end, int64_t *steps_done,
                      double *t_out);

/* Block until all enqueued work of the handle is complete. */
int paraiso_hydro_sync(paraiso_hydro_t *h);

/* Simulation time and number of completed steps.  Blocking.  Either pointer may be NULL. */
int paraiso_hydro_time(paraiso_hydro_t *h, double *t_out, int64_t *steps_out);

/* Number of cell updates whose new state had non-finite values or non-positive rho or p, counted by the
 * last-stage epilogues since set_state.  Blocking.  Returns PARAISO_ENONFINITE if the count is > 0. */
int paraiso_hydro_stats(paraiso_hydro_t *h, int64_t *nonfinite_cells);

/* How many kernels the handle has launched since create (for bench.py's "gpu_launches"). */
int paraiso_hydro_launch_count(paraiso_hydro_t *h, int64_t *launches);

/* Per-stage device timing with CUDA events recorded on the handle's stream around the kernel(s) of every RK
 * stage (for bench.py's roofline: the duration of the dominant kernel inside the timed region).
 *   enable = 1 / 0  switch it on / off and reset the accumulators (blocks until the stream is idle); while on,
 *                   run() launches plainly instead of replaying a graph
 *   enable < 0      read: blocks until the recorded events have completed, then
 *                   *total_ms = summed duration of the timed stages, *stage_launches = how many were timed.
 * Either pointer may be NULL. */
int paraiso_hydro_kernel_time(paraiso_hydro_t *h, int enable, double *total_ms, int64_t *stage_launches);

/* Message for the last error on this handle (or the last create failure when h == NULL).  Never NULL. */
const char *paraiso_hydro_last_error(const paraiso_hydro_t *h);

/* Library version string, e.g. "paraiso_hydro 0.1 sm_100a". */
const char *paraiso_hydro_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PARAISO_HYDRO_H */
