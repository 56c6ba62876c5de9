/* paraiso_wave.h — C ABI of the paper's worked Orthotope-Machine example (§2.3, :250-318):
 * the linear wave equation f_tt = c^2 f_xx as the system (2)-(3), one step = the Paraiso program of Table 2
 * (PAPER.md:289-310):
 *     dx = 2 pi / n ; dt = dx / c                              (periodic on 0 <= x < 2 pi)
 *     f1 = f0 + dt * g0                                        Eq. 6
 *     g1 = g0 + (dt * c^2 / dx^2) * (f1[i-1] + f1[i+1] - 2 * f1[i])          Eq. 7
 *     energy = Reduce Sum 0.5 * (c^2 * ((f1[i+1] - f1[i-1]) / (2 dx))^2 + ((g0 + g1)/2)^2) * dx      Eq. 8 as Table 2 has it
 * It exercises a second stencil and the `Reduce Sum` operator on the same skeleton as the Euler path (one fused kernel
 * per step; the shifted f1 is recomputed, "Delayed"; the sum is a warp-shuffle + block reduction whose per-block
 * partials are added in block order by the last block, so the result does not depend on scheduling).  fp64 (the
 * listing's `Double`), one rounded operation per symbol, no fused multiply-add: bit-equal to the oracle in f and g; the
 * energy differs from a sequential sum only by the summation order.
 * Part of libparaiso_hydro.so.  Return codes: those of paraiso_hydro.h.  Pointers f, g, energy are HOST or DEVICE
 * pointers to n (or nsteps) doubles unless said otherwise; the caller owns them. */
#ifndef PARAISO_WAVE_H
#define PARAISO_WAVE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct paraiso_wave paraiso_wave_t;

/* n >= 3 cells, signal speed c > 0 (3.43 in the paper's runs).  Allocates four arrays of n doubles on the device. */
int paraiso_wave_create(paraiso_wave_t **out, int64_t n, double c);
int paraiso_wave_destroy(paraiso_wave_t *h);
/* f^0 and g^0 (n doubles each).  Blocking. */
int paraiso_wave_set_state(paraiso_wave_t *h, const double *f, const double *g);
int paraiso_wave_get_state(paraiso_wave_t *h, double *f_out, double *g_out);
/* nsteps >= 0 steps; energy_out (HOST pointer, may be NULL) receives the energy of Eq. 8 of each step.  Blocking. */
int paraiso_wave_step(paraiso_wave_t *h, int64_t nsteps, double *energy_out);
/* how many kernels the handle has launched */
int paraiso_wave_launch_count(paraiso_wave_t *h, int64_t *launches);

#ifdef __cplusplus
}
#endif
#endif /* PARAISO_WAVE_H */
