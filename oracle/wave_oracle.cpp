// oracle/wave_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH (same rules as oracle/euler_oracle.cpp: only tests/ may load it;
// no code shared with paper_1204_4779_b200/csrc).
//
// The paper's worked example of an Orthotope Machine program (§2.3, :250-318): the linear wave equation
// f_tt = c^2 f_xx as the first-order system (2)-(3), advanced by the scheme of Eq. 6-7 and monitored through the
// discrete energy of Eq. 8, exactly as the Paraiso source of Table 2 states it — that listing is the
// program that ran, so where Eq. 8 as printed disagrees with it (the factor 1/2 and the place of c^2) the listing is
// followed (R24):
//
//   dx = 2 pi / n ; dt = dx / c                         (0 <= x < 2 pi, periodic; c = 3.43 in the paper's runs)
//   f1 = f0 + dt * g0                                                                    Eq. 6
//   fR = f1[i+1] ; fL = f1[i-1]                         (shift -1 / shift +1 of f1)
//   g1 = g0 + (dt * c^2 / dx^2) * (fL + fR - 2 * f1)                                     Eq. 7
//   dfdx = (fR - fL) / (2 dx)
//   energy = Reduce Sum  0.5 * (c^2 * dfdx^2 + ((g0 + g1)/2)^2) * dx                     Eq. 8 / Table 2
//
// fp64 (the listing's `0::Double`), one rounded operation per symbol, evaluated left to right as written, no fused
// multiply-add; the sum runs over the cells in index order.  Pins (tests/test_oracle_pins.py P17): the paper's own
// statement that the energy fluctuates by less than O(1e-13) for N = 8 .. 3072; the identity
// f^{n+1}[i] + f^{n-1}[i] = f^n[i+1] + f^n[i-1] that Eq. 6-7 satisfy when c dt = dx; hand values on 8 cells.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {
struct Wave {
  int64_t n;
  double c, dx, dt;
  std::vector<double> f, g;
};
}  // namespace

extern "C" {

void* wave_oracle_create(int64_t n, double c) {
  if (n < 3 || !(c > 0)) return nullptr;
  Wave* w = new Wave;
  w->n = n;
  w->c = c;
  w->dx = 2.0 * 3.14159265358979323846 / double(n);
  w->dt = w->dx / c;
  w->f.assign(n, 0.0);
  w->g.assign(n, 0.0);
  return w;
}
void wave_oracle_destroy(void* h) { delete static_cast<Wave*>(h); }
void wave_oracle_set_state(void* h, const double* f, const double* g) {
  Wave* w = static_cast<Wave*>(h);
  std::memcpy(w->f.data(), f, w->n * sizeof(double));
  std::memcpy(w->g.data(), g, w->n * sizeof(double));
}
void wave_oracle_get_state(void* h, double* f, double* g) {
  Wave* w = static_cast<Wave*>(h);
  std::memcpy(f, w->f.data(), w->n * sizeof(double));
  std::memcpy(g, w->g.data(), w->n * sizeof(double));
}
double wave_oracle_dx(void* h) { return static_cast<Wave*>(h)->dx; }
double wave_oracle_dt(void* h) { return static_cast<Wave*>(h)->dt; }

// one step of Table 2; returns the energy of Eq. 8 for this step
double wave_oracle_step(void* h) {
  Wave* w = static_cast<Wave*>(h);
  const int64_t n = w->n;
  const double c = w->c, dx = w->dx, dt = w->dt;
  const double k = dt * (c * c) / (dx * dx);
  std::vector<double> f1(n), g1(n);
  for (int64_t i = 0; i < n; ++i) f1[i] = w->f[i] + dt * w->g[i];
  double energy = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    const double fR = f1[(i + 1) % n];
    const double fL = f1[(i + n - 1) % n];
    g1[i] = w->g[i] + k * (fL + fR - 2.0 * f1[i]);
    const double dfdx = (fR - fL) / (2.0 * dx);
    const double gm = (w->g[i] + g1[i]) / 2.0;
    energy += 0.5 * ((c * c) * (dfdx * dfdx) + gm * gm) * dx;
  }
  w->f.swap(f1);
  w->g.swap(g1);
  return energy;
}

}  // extern "C"
