/* paraiso_hydro_noalloc.h — the CFL time step of a state the caller already holds on the device, computed without a
 * single device or host allocation by this library.  Exported by libparaiso_hydro.so; return codes are those of
 * paraiso_hydro.h plus PARAISO_ETOOLARGE below.
 *
 * Who this is for.  Everything else in the library goes through a handle, and paraiso_hydro_create() allocates: two
 * copies of the state plus the control block.  Some users of a hydro step cannot accept that:
 *   - a simulation code that has handed the whole of HBM to its own arena (or to a framework's caching allocator) at
 *     start-up.  A 512^3 run keeps 2.7 GB per state copy; a cudaMalloc from a plug-in either fails there or takes
 *     memory the host code has budgeted for something else;
 *   - an in-situ tool (a monitor, a load balancer, a coupling layer) that is only lent a pointer to somebody else's
 *     state between two of their kernels and must leave the device's memory map exactly as it found it;
 *   - a time-step loop that must never stall: cudaMalloc and cudaFree synchronise the whole device, so a call that
 *     may allocate cannot sit between asynchronously queued stages.
 * Such callers get ONE entry point that needs no handle: paraiso_hydro_cfl_noalloc(), the reduction S = max over
 * cells and axes of (|v_a| + c) / dr_a and dt = cfl / S ("the time step determined by the
 * CFL-condition"; R6), i.e. what paraiso_hydro_cfl_dt() returns for a handle holding the same state.
 *
 * Where its working memory lives.  The reduction needs one partial maximum and one bad-cell count per thread block
 * and a ticket that tells the last block it is the last.  Instead of a cudaMalloc'ed buffer these sit in a fixed
 * array compiled into the library (PARAISO_NOALLOC_SCRATCH_BYTES of device memory, reserved on every GPU on which the
 * library's code is loaded, until the process exits).  That fixed size is what bounds the grid: at most
 * PARAISO_NOALLOC_MAX_CELLS cells.
 */
#ifndef PARAISO_HYDRO_NOALLOC_H
#define PARAISO_HYDRO_NOALLOC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* One block reduces 4096 cells; the scratch has room for 32768 blocks: 2^27 cells = 512^3 (config 4). */
#define PARAISO_NOALLOC_MAX_CELLS 134217728LL
/* 256-byte header (the ticket) + 32768 x (8-byte partial maximum + 4-byte bad-cell count) */
#define PARAISO_NOALLOC_SCRATCH_BYTES 393472
/* returned when the grid has more than PARAISO_NOALLOC_MAX_CELLS cells: the built-in scratch cannot hold its partials
 * (a code of its own, next to those of paraiso_hydro.h, so that the caller can tell it from a malformed argument) */
#define PARAISO_ETOOLARGE (-6)

/* S, dt and the bad-cell count of a conserved state U, with no allocation.
 *   dims, n[dims], extent[dims], gamma, dtype   as for paraiso_hydro_create (x first; n[a] >= 1 here, no stencil)
 *   U_dev     DEVICE pointer, caller-owned, read only: (dims+2) * N elements of `dtype`, SoA, field-major, x fastest
 *             (rho, m_x[, m_y[, m_z]], E), N = prod n[a].  It must be on the current device.
 *   cfl       finite, > 0
 *   cuda_stream  a cudaStream_t of the current device (NULL = the legacy default stream); all work is queued on it
 *   out_dev   DEVICE pointer, caller-owned, 3 doubles, written by the kernel:
 *               out_dev[0] = S (widened exactly from `dtype`),
 *               out_dev[1] = dt = Real(cfl) / S, one IEEE division in `dtype` (the same division cfl_dt performs),
 *               out_dev[2] = number of cells with rho or p not > 0 or a non-finite E (they never raise S).
 * Asynchronous: returns once the work is queued; read out_dev after the stream has caught up.
 *
 * Errors: PARAISO_EINVAL for a null pointer, dims outside 1..3, n[a] < 1, gamma <= 1, a bad cfl or dtype;
 * PARAISO_ETOOLARGE for N > PARAISO_NOALLOC_MAX_CELLS (use a handle for larger grids, or reduce sub-boxes and take
 * the larger S); PARAISO_ECUDA when there is no device or a CUDA call fails.  Nothing is queued when an error is
 * returned.
 *
 * What the caller has to know:
 *   - This function calls no cudaMalloc, cudaFree or other allocating routine, on any call.
 *   - The FIRST call on each device looks up the device address of the built-in scratch array (and the CUDA runtime
 *     loads the kernel then).  Make that first call during set-up, with the device current, before any stream
 *     capture is begun; later calls on that device only queue a 256-byte memset and one kernel.
 *   - All calls on one device share the one scratch array, whatever their streams.  The array still holds the
 *     previous call's partial results; the function clears the part that must start at zero (the ticket) on the
 *     given stream before the kernel.  Two calls that can overlap on the GPU (different streams without an event
 *     between them, or two host threads) race on the scratch and give wrong answers: order them.
 *   - Thread safety: the first-call set-up is guarded; the scratch itself is not (previous point).
 */
int paraiso_hydro_cfl_noalloc(int dims, const int64_t *n, const double *extent, double gamma, int dtype,
                              const void *U_dev, double cfl, void *cuda_stream, double *out_dev);

#ifdef __cplusplus
}
#endif
#endif /* PARAISO_HYDRO_NOALLOC_H */
