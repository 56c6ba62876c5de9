// oracle/euler_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT PART OF THE PRODUCT PATH.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this file's shared object.  It shares no code with paper_1204_4779_b200/csrc (the CUDA
// path): no common header, helper, table or constant generator.
//
// What it is: a plain, slow, single-threaded (optionally OpenMP over independent cells, results
// bit-identical) restatement of ONE explicit time step of the finite-volume compressible Euler
// solver of PAPER.md §4.1, plus the global CFL reduction that sets dt
// (PAPER.md:25, 736).  The method is an explicit scheme with no independent "plain definition" of
// its result, so this file follows the algorithm step by step, in the paper's order and notation:
//
//   Eq. 19  V0 = V(U0)                               -> prim_of()
//   Eq. 20  (VR[i-1/2], VL[i+1/2]) = Interpolate()   -> minbee() applied per primitive field
//   Eq. 21  MINBEE limiter, literal order of cases   -> minbee()
//   Eq. 22  F_a[i+1/2] = HLLC_a(VL, VR)              -> riemann()  (HLL selectable, R4)
//   Eq. 23  AddFlux                                  -> stage()
//   Eq. 24-27 two-stage (midpoint) time marching     -> step()
//
// Readings of the paper where it is silent or garbled are listed in DESIGN.md §3 (R1..R19); the
// written arithmetic (operation order and the places where a fused multiply-add is used) is
// DESIGN.md §4 and is part of the specification: the CUDA path states the same order, so that the
// two can agree to the last bit.  No floors, positivity fixes or entropy fixes: the paper has none.
//
// Pins (tests/test_oracle_pins.py, `-m "not gpu"`): uniform state bitwise fixed (P1), conservation
// (P2), closed-form first half-stage of the N=8 Sod problem for HLL and HLLC (P3, values in
// tests/golden/sod_n8_first_stage.txt), stationary contact (P4), Sod against the exact Riemann
// solution (P5), the paper's entropy-wave and sound-wave tests Eq. 28-29 with ~2nd-order
// convergence (P6, P7), x/y/z embedding identity (P8), mirror symmetry (P9), Riemann-solver
// special cases (P10), an independent NumPy restatement on <= 8 cells (P11), primitive <-> conserved
// conversion against closed forms and its round trip (P13).
// Every exported function below is pinned by at least one of these; nothing here is "parity
// unpinned".  (Unpinned, because absent from the text: the error curves of the paper's Fig. 10.)
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -mfma -shared -fPIC   (see oracle/build.py)
//   -ffp-contract=off : no implicit contraction; std::fma appears only where DESIGN.md §4 writes fma
//   -mfma             : std::fma compiles to the hardware instruction (correctly rounded either way)

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { BOUNDARY_PERIODIC = 0, BOUNDARY_OUTFLOW = 1 };
enum { RIEMANN_HLLC = 0, RIEMANN_HLL = 1 };
// Interpolation variants ("interpolation methods ... combinable"): the paper's
// MINBEE (Eq. 21, the default and what every BASELINE config runs), none (dy = 0: piecewise-constant states, the
// first-order Godunov scheme) and the monotonized-central limiter (van Leer 1977, "MC"), an option like HLL.
enum { LIMITER_MINBEE = 0, LIMITER_NONE = 1, LIMITER_MC = 2 };

// Primitive variables V = (rho, v_a, p), Eq. 13.  Components b >= D are zero.
template <class Real>
struct Prim {
  Real rho, v[3], p;
};

template <class Real, int D>
struct Solver {
  static constexpr int NF = D + 2;  // d+2 degrees of freedom

  int64_t n[3];  // cells per axis, x first; n[a] = 1 for a >= D
  int64_t N;     // total cells
  Real dr[3];    // mesh size  dr_a = Real(extent_a / n_a)   (Eq. 23 "Delta r_a")
  Real idr[3];   // Real(n_a / extent_a), used only by the CFL reduction (R6)
  Real gamma, gm1, igm1;
  int boundary = BOUNDARY_PERIODIC;
  int riemann_kind = RIEMANN_HLLC;
  std::vector<Real> U;  // conserved state, SoA: U[f*N + (k*n1 + j)*n0 + i], f = rho, m_x.., E
  double t = 0.0;

  Solver(const int64_t* n_, const double* extent, double gamma_) {
    N = 1;
    for (int a = 0; a < 3; ++a) {
      n[a] = a < D ? n_[a] : 1;
      N *= n[a];
      dr[a] = a < D ? Real(extent[a] / double(n[a])) : Real(1);
      idr[a] = a < D ? Real(double(n[a]) / extent[a]) : Real(0);
    }
    gamma = Real(gamma_);
    gm1 = gamma - Real(1);
    igm1 = Real(1) / gm1;
    U.assign(size_t(NF) * N, Real(0));
  }

  // ghost cells: periodic = index wrap; outflow = index clamp (R12)
  int64_t map_index(int64_t i, int64_t na) const {
    if (boundary == BOUNDARY_PERIODIC) {
      int64_t r = i % na;
      return r < 0 ? r + na : r;
    }
    return i < 0 ? 0 : (i >= na ? na - 1 : i);
  }
  int64_t cell(int64_t i, int64_t j, int64_t k) const { return (k * n[1] + j) * n[0] + i; }

  // Eq. 19 with the ideal-gas EOS E = p/(gamma-1) + rho v^2/2.
  Prim<Real> prim_of(const Real* Uc, int64_t c) const {
    Prim<Real> V;
    const Real rho = Uc[c];
    const Real ir = Real(1) / rho;
    Real q = Real(0);
    for (int b = 0; b < 3; ++b) {
      V.v[b] = b < D ? Uc[size_t(1 + b) * N + c] * ir : Real(0);
      if (b == 0)
        q = V.v[0] * V.v[0];
      else if (b < D)
        q = std::fma(V.v[b], V.v[b], q);
    }
    const Real E = Uc[size_t(D + 1) * N + c];
    V.rho = rho;
    V.p = gm1 * std::fma(-(Real(0.5) * rho), q, E);
    return V;
  }

  // The inverse of Eq. 19: U = (rho, rho v_a, E) with the EOS E = p/(gamma-1) + rho v^2/2, written
  // as in DESIGN.md §4 "cons": q as in prim_of, E = fma(0.5 rho, q, p igm1).  Used when a caller hands over
  // primitive variables (state_kind = 1 of the C ABI); pinned by closed-form values and the round trip (P13).
  void set_primitive(const Real* V) {
    for (int64_t c = 0; c < N; ++c) {
      const Real rho = V[c];
      Real q = Real(0);
      for (int b = 0; b < D; ++b) {
        const Real vb = V[size_t(1 + b) * N + c];
        q = b == 0 ? vb * vb : std::fma(vb, vb, q);
        U[size_t(1 + b) * N + c] = rho * vb;
      }
      U[c] = rho;
      U[size_t(D + 1) * N + c] = std::fma(Real(0.5) * rho, q, V[size_t(D + 1) * N + c] * igm1);
    }
    t = 0.0;
  }
  void get_primitive(Real* V) const {
    for (int64_t c = 0; c < N; ++c) {
      const Prim<Real> P = prim_of(U.data(), c);
      V[c] = P.rho;
      for (int b = 0; b < D; ++b) V[size_t(1 + b) * N + c] = P.v[b];
      V[size_t(D + 1) * N + c] = P.p;
    }
  }

  // Eq. 21, literal order of the three cases (R9).
  static void minbee(Real y0, Real y1, Real y2, Real& lo, Real& hi) {
    const Real d01 = y1 - y0;
    const Real d12 = y2 - y1;
    Real dy;
    if (d01 * d12 < Real(0))
      dy = Real(0);
    else if (std::fabs(d01) < std::fabs(d12))
      dy = d01;
    else
      dy = d12;
    lo = std::fma(Real(-0.5), dy, y1);  // y1 - dy/2   (face i-1/2 side)
    hi = std::fma(Real(0.5), dy, y1);   // y1 + dy/2   (face i+1/2 side)
  }

  // Options beside Eq. 21 (R22), same form (lo, hi) = (y1 - dy/2, y1 + dy/2):
  //   none: dy = 0 (the scheme degenerates to first-order Godunov, pin P10/P15)
  //   MC  : dy = 0 if dy01 * dy12 < 0 (the same product test as Eq. 21), else the value of smallest magnitude among
  //         2 dy01, 2 dy12 and the central difference dc = (dy01 + dy12)/2, with the sign of dc
  static void limited(int lim, Real y0, Real y1, Real y2, Real& lo, Real& hi) {
    if (lim == LIMITER_MINBEE) {
      minbee(y0, y1, y2, lo, hi);
      return;
    }
    Real dy = Real(0);
    if (lim == LIMITER_MC) {
      const Real d01 = y1 - y0;
      const Real d12 = y2 - y1;
      const Real dc = Real(0.5) * (d01 + d12);
      const Real a = std::fmin(std::fmin(Real(2) * std::fabs(d01), Real(2) * std::fabs(d12)), std::fabs(dc));
      dy = (d01 * d12 < Real(0)) ? Real(0) : std::copysign(a, dc);
    }
    lo = std::fma(Real(-0.5), dy, y1);
    hi = std::fma(Real(0.5), dy, y1);
  }

  // Interpolate (Eq. 20) applied to a whole primitive state, component by component.
  int limiter = LIMITER_MINBEE;
  void interpolate(const Prim<Real>& V0, const Prim<Real>& V1, const Prim<Real>& V2,
                   Prim<Real>& lo, Prim<Real>& hi) const {
    limited(limiter, V0.rho, V1.rho, V2.rho, lo.rho, hi.rho);
    for (int b = 0; b < 3; ++b) {
      if (b < D)
        limited(limiter, V0.v[b], V1.v[b], V2.v[b], lo.v[b], hi.v[b]);
      else
        lo.v[b] = hi.v[b] = Real(0);
    }
    limited(limiter, V0.p, V1.p, V2.p, lo.p, hi.p);
  }

  // Eq. 22: flux through a face with normal e_a from the left/right primitive states.
  // HLLC: Toro, Spruce & Speares (ref [32]) as restated in Toro's textbook (ref [30]) section 10.4;
  // HLL: same wave-speed estimates.  Wave speeds: Davis (R5).  F[f], f = rho, m_b.., E.
  void riemann(int a, const Prim<Real>& L, const Prim<Real>& R, Real* F) const {
    const Prim<Real>* K2[2] = {&L, &R};
    Real c[2], q[2], E[2], m[2], UK[2][5], FK[2][5];
    for (int s = 0; s < 2; ++s) {
      const Prim<Real>& K = *K2[s];
      c[s] = std::sqrt((gamma * K.p) / K.rho);
      q[s] = K.v[0] * K.v[0];
      for (int b = 1; b < D; ++b) q[s] = std::fma(K.v[b], K.v[b], q[s]);
      E[s] = std::fma(Real(0.5) * K.rho, q[s], K.p * igm1);
      m[s] = K.rho * K.v[a];  // mass flux rho v_a (R2)
      UK[s][0] = K.rho;
      FK[s][0] = m[s];
      for (int b = 0; b < D; ++b) {
        UK[s][1 + b] = K.rho * K.v[b];
        FK[s][1 + b] = (b == a) ? std::fma(m[s], K.v[b], K.p) : m[s] * K.v[b];  // Eq. 15
      }
      UK[s][D + 1] = E[s];
      FK[s][D + 1] = K.v[a] * (E[s] + K.p);
    }
    const Real vnL = L.v[a], vnR = R.v[a];
    const Real SL = std::fmin(vnL - c[0], vnR - c[1]);
    const Real SR = std::fmax(vnL + c[0], vnR + c[1]);
    if (SL >= Real(0)) {
      for (int f = 0; f < NF; ++f) F[f] = FK[0][f];
      return;
    }
    if (SR <= Real(0)) {
      for (int f = 0; f < NF; ++f) F[f] = FK[1][f];
      return;
    }
    if (riemann_kind == RIEMANN_HLL) {
      const Real inv = Real(1) / (SR - SL);
      const Real SLSR = SL * SR;
      for (int f = 0; f < NF; ++f) {
        // (SR FL - SL FR + SL SR (UR - UL)) / (SR - SL)
        const Real num = std::fma(SLSR, UK[1][f] - UK[0][f], std::fma(SR, FK[0][f], -(SL * FK[1][f])));
        F[f] = num * inv;
      }
      return;
    }
    const Real aL = L.rho * (SL - vnL);
    const Real aR = R.rho * (SR - vnR);
    const Real Sstar = std::fma(-aR, vnR, std::fma(aL, vnL, R.p - L.p)) / (aL - aR);
    const int s = (Sstar >= Real(0)) ? 0 : 1;  // upwind side K (R10)
    const Prim<Real>& K = *K2[s];
    const Real SK = s == 0 ? SL : SR;
    const Real aK = s == 0 ? aL : aR;
    const Real vnK = K.v[a];
    const Real fK = aK / (SK - Sstar);  // rho*_K
    Real Ustar[5];
    Ustar[0] = fK;
    for (int b = 0; b < D; ++b) Ustar[1 + b] = (b == a) ? fK * Sstar : fK * K.v[b];
    Ustar[D + 1] = fK * std::fma(Sstar - vnK, Sstar + K.p / aK, E[s] / K.rho);
    for (int f = 0; f < NF; ++f) F[f] = std::fma(SK, Ustar[f] - UK[s][f], FK[s][f]);  // F*K = FK + SK(U*K - UK)
  }

  // One stage:  U_out = AddFlux(tau, Flux_a(U_in), U_base), Eq. 23-27.
  // The sum over axes runs x, y, z, accumulated left to right onto U_base (R11).
  void stage(const std::vector<Real>& Uin, const std::vector<Real>& Ubase, Real tau,
             std::vector<Real>& Uout) const {
    std::vector<Prim<Real>> V(N);
#pragma omp parallel for
    for (int64_t c = 0; c < N; ++c) V[c] = prim_of(Uin.data(), c);

    Uout = Ubase;
    for (int a = 0; a < D; ++a) {
      const Real lambda = tau / dr[a];
      const int64_t na = n[a];
      // line(l) enumerates the cells of one grid line along axis a: cell index = base + i*stride
      const int64_t stride = a == 0 ? 1 : (a == 1 ? n[0] : n[0] * n[1]);
      const int64_t nlines = N / na;
#pragma omp parallel for
      for (int64_t l = 0; l < nlines; ++l) {
        int64_t base;
        if (a == 0)
          base = l * n[0];
        else if (a == 1)
          base = (l / n[0]) * n[0] * n[1] + (l % n[0]);
        else
          base = l;
        // fluxes at faces f+1/2, f = -1 .. na-1, stored at Fl[(f+1)*NF + field]
        std::vector<Real> Fl(size_t(na + 1) * NF);
        for (int64_t f = -1; f < na; ++f) {
          const Prim<Real>& Vm = V[base + map_index(f - 1, na) * stride];
          const Prim<Real>& V0 = V[base + map_index(f, na) * stride];
          const Prim<Real>& V1 = V[base + map_index(f + 1, na) * stride];
          const Prim<Real>& V2 = V[base + map_index(f + 2, na) * stride];
          Prim<Real> lo0, hi0, lo1, hi1;
          interpolate(Vm, V0, V1, lo0, hi0);  // cell f   : its hi is VL[f+1/2]
          interpolate(V0, V1, V2, lo1, hi1);  // cell f+1 : its lo is VR[f+1/2]
          riemann(a, hi0, lo1, &Fl[size_t(f + 1) * NF]);
        }
        for (int64_t i = 0; i < na; ++i) {
          const int64_t c = base + i * stride;
          for (int f = 0; f < NF; ++f) {
            const Real dF = Fl[size_t(i) * NF + f] - Fl[size_t(i + 1) * NF + f];  // F[i-1/2] - F[i+1/2]
            Uout[size_t(f) * N + c] = std::fma(lambda, dF, Uout[size_t(f) * N + c]);
          }
        }
      }
    }
  }

  // Eq. 24-27 (midpoint form, R7) -- the paper's integrator, the default.
  // integrator = 1: the two-stage TVD Runge-Kutta scheme north_star names as the fallback (Heun / Shu-Osher
  // SSP-RK2, R20):  U1 = U0 + dt L(U0);  U2 = 0.5 (U0 + (U1 + dt L(U1))).  An option, never the default.
  int integrator = 0;
  void step(Real dt) {
    std::vector<Real> U1, U2;
    if (integrator == 0) {
      stage(U, U, Real(0.5) * dt, U1);
      stage(U1, U, dt, U2);
    } else {
      stage(U, U, dt, U1);
      stage(U1, U1, dt, U2);
      for (size_t i = 0; i < U2.size(); ++i) U2[i] = Real(0.5) * (U[i] + U2[i]);
    }
    U.swap(U2);
  }

  // Prescribed ghost cells ("we substitute the analytic solutions to the ghost
  // cells"): the outermost two cells of every axis ARE the ghost cells of this mode (two = the stencil reach of Eq.
  // 20-22).  The caller overwrites them with its own values G (an array shaped like the state, of which only those
  // cells are read) before a step and between the two stages; the cells in between are advanced by Eq. 23-27 as
  // always, and what the scheme computes in the ghost cells themselves (with the clamped index of the outflow mode)
  // is overwritten before anything reads it (R23).
  bool in_frame(int64_t c) const {
    int64_t idx[3] = {c % n[0], (c / n[0]) % n[1], c / (n[0] * n[1])};
    for (int a = 0; a < D; ++a)
      if (idx[a] < 2 || idx[a] >= n[a] - 2) return true;
    return false;
  }
  void inject_frame(std::vector<Real>& A, const Real* G) const {
    for (int64_t c = 0; c < N; ++c)
      if (in_frame(c))
        for (int f = 0; f < NF; ++f) A[size_t(f) * N + c] = G[size_t(f) * N + c];
  }
  void step_ghosts(Real dt, const Real* Gmid) {
    std::vector<Real> U1, U2;
    if (integrator == 0) {
      stage(U, U, Real(0.5) * dt, U1);
      inject_frame(U1, Gmid);
      stage(U1, U, dt, U2);
    } else {
      stage(U, U, dt, U1);
      inject_frame(U1, Gmid);
      stage(U1, U1, dt, U2);
      for (size_t i = 0; i < U2.size(); ++i) U2[i] = Real(0.5) * (U[i] + U2[i]);
    }
    U.swap(U2);
  }

  // S = max_cells max_a (|v_a| + c) / dr_a   (R6);  dt = Real(cfl) / S.
  Real cfl_S() const {
    Real S = Real(0);
#pragma omp parallel for reduction(max : S)
    for (int64_t c = 0; c < N; ++c) {
      const Prim<Real> V = prim_of(U.data(), c);
      const Real ir = Real(1) / V.rho;
      const Real cs = std::sqrt((gamma * V.p) * ir);
      Real s = Real(0);
      for (int a = 0; a < D; ++a) s = std::fmax(s, (std::fabs(V.v[a]) + cs) * idr[a]);
      S = std::fmax(S, s);
    }
    return S;
  }
};

struct Handle {
  int dims, dtype;
  void* solver;
};

template <class F>
auto dispatch(const Handle* h, F&& f) {
  if (h->dtype == 0) {
    if (h->dims == 1) return f(static_cast<Solver<float, 1>*>(h->solver));
    if (h->dims == 2) return f(static_cast<Solver<float, 2>*>(h->solver));
    return f(static_cast<Solver<float, 3>*>(h->solver));
  }
  if (h->dims == 1) return f(static_cast<Solver<double, 1>*>(h->solver));
  if (h->dims == 2) return f(static_cast<Solver<double, 2>*>(h->solver));
  return f(static_cast<Solver<double, 3>*>(h->solver));
}

template <class Real, int D>
void riemann_probe(int a, int kind, double gamma, const double* VL, const double* VR, double* F) {
  const int64_t n[3] = {4, 4, 4};
  const double ext[3] = {1, 1, 1};
  Solver<Real, D> s(n, ext, gamma);
  s.riemann_kind = kind;
  Prim<Real> L{}, R{};
  L.rho = Real(VL[0]);
  R.rho = Real(VR[0]);
  for (int b = 0; b < D; ++b) {
    L.v[b] = Real(VL[1 + b]);
    R.v[b] = Real(VR[1 + b]);
  }
  L.p = Real(VL[D + 1]);
  R.p = Real(VR[D + 1]);
  Real Fr[5];
  s.riemann(a, L, R, Fr);
  for (int f = 0; f < D + 2; ++f) F[f] = double(Fr[f]);
}

}  // namespace

extern "C" {

// dtype: 0 = float, 1 = double.  n[dims] x first, extent[dims] physical lengths.
void* oracle_create(int dims, const int64_t* n, const double* extent, double gamma, int dtype) {
  if (dims < 1 || dims > 3 || (dtype != 0 && dtype != 1)) return nullptr;
  Handle* h = new Handle{dims, dtype, nullptr};
  if (dtype == 0) {
    if (dims == 1) h->solver = new Solver<float, 1>(n, extent, gamma);
    if (dims == 2) h->solver = new Solver<float, 2>(n, extent, gamma);
    if (dims == 3) h->solver = new Solver<float, 3>(n, extent, gamma);
  } else {
    if (dims == 1) h->solver = new Solver<double, 1>(n, extent, gamma);
    if (dims == 2) h->solver = new Solver<double, 2>(n, extent, gamma);
    if (dims == 3) h->solver = new Solver<double, 3>(n, extent, gamma);
  }
  return h;
}

void oracle_destroy(void* hv) {
  Handle* h = static_cast<Handle*>(hv);
  if (!h) return;
  dispatch(h, [](auto* s) {
    delete s;
    return 0;
  });
  delete h;
}

// key: "boundary" (0 periodic, 1 outflow) | "riemann" (0 HLLC, 1 HLL) | "integrator" (0 midpoint, 1 Heun) |
//      "limiter" (0 MINBEE, 1 none, 2 MC)
int oracle_set_option(void* hv, const char* key, int64_t value) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    if (!std::strcmp(key, "boundary") && (value == 0 || value == 1)) {
      s->boundary = int(value);
      return 0;
    }
    if (!std::strcmp(key, "riemann") && (value == 0 || value == 1)) {
      s->riemann_kind = int(value);
      return 0;
    }
    if (!std::strcmp(key, "integrator") && (value == 0 || value == 1)) {
      s->integrator = int(value);
      return 0;
    }
    if (!std::strcmp(key, "limiter") && value >= 0 && value <= 2) {
      s->limiter = int(value);
      return 0;
    }
    return -1;
  });
}

int oracle_set_state(void* hv, const void* U) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    std::memcpy(s->U.data(), U, s->U.size() * sizeof(s->U[0]));
    s->t = 0.0;
    return 0;
  });
}

int oracle_get_state(void* hv, void* U) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    std::memcpy(U, s->U.data(), s->U.size() * sizeof(s->U[0]));
    return 0;
  });
}

int oracle_set_primitive(void* hv, const void* V) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    s->set_primitive(static_cast<const Real*>(V));
    return 0;
  });
}

int oracle_get_primitive(void* hv, void* V) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    s->get_primitive(static_cast<Real*>(V));
    return 0;
  });
}

// dt = Real(cfl) / S of the current state, returned widened to double.
double oracle_cfl_dt(void* hv, double cfl) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    return double(Real(cfl) / s->cfl_S());
  });
}

// one full RK2 step with dt rounded to the handle's precision
int oracle_step(void* hv, double dt) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    s->step(Real(dt));
    s->t += double(Real(dt));
    return 0;
  });
}

// Prescribed ghost cells: overwrite the outermost two cells of every axis of the current state with G's
int oracle_set_ghosts(void* hv, const void* G) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    s->inject_frame(s->U, static_cast<const Real*>(G));
    return 0;
  });
}

// one full RK2 step; the ghost cells of the intermediate state U1 are overwritten with Gmid's before the second stage
int oracle_step_ghosts(void* hv, double dt, const void* Gmid) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    s->step_ghosts(Real(dt), static_cast<const Real*>(Gmid));
    s->t += double(Real(dt));
    return 0;
  });
}

// Uout = AddFlux(tau, Flux(U), U): one stage applied to the current state, which is not modified.
int oracle_stage(void* hv, double tau, void* Uout) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    std::vector<Real> out;
    s->stage(s->U, s->U, Real(tau), out);
    std::memcpy(Uout, out.data(), out.size() * sizeof(Real));
    return 0;
  });
}

// Advance with dt from the CFL condition at the start of every step (R6), for nsteps
// steps or until t_end (> 0) is reached, the last step clamped to land on t_end (R18).
int oracle_run(void* hv, double cfl, int64_t nsteps, double t_end, int64_t* steps_done, double* t_out) {
  Handle* h = static_cast<Handle*>(hv);
  return dispatch(h, [&](auto* s) {
    using Real = std::decay_t<decltype(s->gamma)>;
    int64_t k = 0;
    for (; k < nsteps; ++k) {
      if (t_end > 0.0 && s->t >= t_end) break;
      Real dt = Real(cfl) / s->cfl_S();
      bool last = false;
      if (t_end > 0.0 && s->t + double(dt) >= t_end) {
        dt = Real(t_end - s->t);
        last = true;
      }
      s->step(dt);
      s->t = last ? t_end : s->t + double(dt);
    }
    if (steps_done) *steps_done = k;
    if (t_out) *t_out = s->t;
    return 0;
  });
}

// Probes for the pins: one Riemann solve / one limiter evaluation in the requested precision.
// VL, VR: (rho, v_x[, v_y[, v_z]], p) as doubles; F: dims+2 doubles.
int oracle_riemann(int dtype, int dims, int axis, int kind, double gamma, const double* VL,
                   const double* VR, double* F) {
  if (dims < 1 || dims > 3 || axis < 0 || axis >= dims) return -1;
  if (dtype == 0) {
    if (dims == 1) riemann_probe<float, 1>(axis, kind, gamma, VL, VR, F);
    if (dims == 2) riemann_probe<float, 2>(axis, kind, gamma, VL, VR, F);
    if (dims == 3) riemann_probe<float, 3>(axis, kind, gamma, VL, VR, F);
  } else {
    if (dims == 1) riemann_probe<double, 1>(axis, kind, gamma, VL, VR, F);
    if (dims == 2) riemann_probe<double, 2>(axis, kind, gamma, VL, VR, F);
    if (dims == 3) riemann_probe<double, 3>(axis, kind, gamma, VL, VR, F);
  }
  return 0;
}

int oracle_minbee(int dtype, double y0, double y1, double y2, double* lo, double* hi) {
  if (dtype == 0) {
    float l, h;
    Solver<float, 1>::minbee(float(y0), float(y1), float(y2), l, h);
    *lo = l;
    *hi = h;
  } else {
    Solver<double, 1>::minbee(y0, y1, y2, *lo, *hi);
  }
  return 0;
}

// one evaluation of an interpolation variant (limiter: 0 MINBEE, 1 none, 2 MC) in the requested precision
int oracle_limited(int dtype, int limiter, double y0, double y1, double y2, double* lo, double* hi) {
  if (limiter < 0 || limiter > 2) return -1;
  if (dtype == 0) {
    float l, h;
    Solver<float, 1>::limited(limiter, float(y0), float(y1), float(y2), l, h);
    *lo = l;
    *hi = h;
  } else {
    Solver<double, 1>::limited(limiter, y0, y1, y2, *lo, *hi);
  }
  return 0;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
