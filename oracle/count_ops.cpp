// count_ops.cpp — TEST / MEASUREMENT INFRASTRUCTURE (like everything under oracle/): a mechanical count of the
// arithmetic of one Euler step (Eq. 19-27), obtained by instantiating the oracle's own Solver with a
// scalar type that tallies every operation it performs ("instantiate the oracle with a CountingReal").
// The oracle source is included unchanged; nothing here alters its arithmetic, and the values a Counting<Base> carries
// are plain Base values, so every data-dependent branch (MINBEE cases, supersonic faces, the upwind side) is taken
// exactly as in the fp32 / fp64 run.  Built without OpenMP (the pragmas are ignored; the tallies are plain globals).
//
// Two counts come out of it (tests/count_ops.py turns them into the committed table):
//   as_written : cfl_S() + step() run whole.  The oracle forms both faces' interpolations per face (every cell is
//                interpolated twice per axis) and both sides' U_K, F_K before the upwind test, as DESIGN.md §4 writes it.
//   composed   : the same member functions called piece by piece on the same data and put together as a kernel that
//                keeps intermediates would: per cell and stage one prim_of, per axis ONE interpolate and one riemann,
//                the Eq. 23 update; per step two stages plus the CFL term.  Still both sides formed in riemann.
#include <cstdint>

struct OpTally {
  uint64_t add, mul, fma, div, sqrt, cmp, minmax, abs, neg, copysign;
};
static OpTally g_tally;

template <class Base>
struct Counting {
  Base v;
  Counting() : v(0) {}
  Counting(double x) : v(Base(x)) {}  // conversions are not arithmetic: not counted
  explicit operator double() const { return double(v); }
  explicit operator float() const { return float(v); }
  friend Counting operator+(Counting a, Counting b) { ++g_tally.add; return Counting(a.v + b.v, 0); }
  friend Counting operator-(Counting a, Counting b) { ++g_tally.add; return Counting(a.v - b.v, 0); }
  friend Counting operator*(Counting a, Counting b) { ++g_tally.mul; return Counting(a.v * b.v, 0); }
  friend Counting operator/(Counting a, Counting b) { ++g_tally.div; return Counting(a.v / b.v, 0); }
  friend Counting operator-(Counting a) { ++g_tally.neg; return Counting(-a.v, 0); }
  friend bool operator<(Counting a, Counting b) { ++g_tally.cmp; return a.v < b.v; }
  friend bool operator>(Counting a, Counting b) { ++g_tally.cmp; return a.v > b.v; }
  friend bool operator<=(Counting a, Counting b) { ++g_tally.cmp; return a.v <= b.v; }
  friend bool operator>=(Counting a, Counting b) { ++g_tally.cmp; return a.v >= b.v; }
  Counting(Base x, int) : v(x) {}  // exact carrier of a result
};

#include <cmath>
namespace std {  // the oracle calls these std::-qualified; overloads for the counting type only (test tool)
template <class B> Counting<B> fma(Counting<B> a, Counting<B> b, Counting<B> c) { ++g_tally.fma; return Counting<B>(std::fma(a.v, b.v, c.v), 0); }
template <class B> Counting<B> sqrt(Counting<B> a) { ++g_tally.sqrt; return Counting<B>(std::sqrt(a.v), 0); }
template <class B> Counting<B> fabs(Counting<B> a) { ++g_tally.abs; return Counting<B>(std::fabs(a.v), 0); }
template <class B> Counting<B> fmin(Counting<B> a, Counting<B> b) { ++g_tally.minmax; return Counting<B>(std::fmin(a.v, b.v), 0); }
template <class B> Counting<B> fmax(Counting<B> a, Counting<B> b) { ++g_tally.minmax; return Counting<B>(std::fmax(a.v, b.v), 0); }
template <class B> Counting<B> copysign(Counting<B> a, Counting<B> b) { ++g_tally.copysign; return Counting<B>(std::copysign(a.v, b.v), 0); }
}  // namespace std

#include "euler_oracle.cpp"  // the oracle, unchanged (its anonymous namespace is visible in this translation unit)

namespace {

constexpr int NCLASS = 10;
void store(const OpTally& t, uint64_t* out) {
  const uint64_t v[NCLASS] = {t.add, t.mul, t.fma, t.div, t.sqrt, t.cmp, t.minmax, t.abs, t.neg, t.copysign};
  for (int i = 0; i < NCLASS; ++i) out[i] = v[i];
}

// out[0..9]   as_written: one cfl_S() + one step(dt), whole grid
// out[10..19] composed: prim_of per cell, ONE interpolate per cell and axis, one riemann per face, update, x 2 stages,
//             + the CFL term (prim_of + speed) once per cell; faces and cells of the state at the start of the step
//             (stage 1) and of U1 (stage 2)
template <class Base, int D>
void count(const int64_t* n, const double* extent, double gamma, int boundary, int riemann_kind, const Base* U0,
           double cfl, uint64_t* out) {
  using R = Counting<Base>;
  Solver<R, D> s(n, extent, gamma);
  s.boundary = boundary;
  s.riemann_kind = riemann_kind;
  constexpr int NF = D + 2;
  for (size_t i = 0; i < size_t(NF) * s.N; ++i) s.U[i] = R(U0[i], 0);

  // ---- as written
  g_tally = OpTally{};
  const R S = s.cfl_S();
  const R dt = R(Base(cfl), 0) / S;
  const std::vector<R> Ustart = s.U;
  std::vector<R> U1;
  {
    Solver<R, D> probe = s;
    probe.stage(probe.U, probe.U, R(0.5) * dt, U1);  // U1 for the composed count of stage 2 (tallied, reset below)
  }
  g_tally = OpTally{};
  (void)s.cfl_S();
  {
    const R dt2 = R(Base(cfl), 0) / S;  // the one division of cfl_dt, part of the step's work
    s.step(dt2);
  }
  store(g_tally, out);

  // ---- composed
  g_tally = OpTally{};
  Solver<R, D> c(n, extent, gamma);
  c.boundary = boundary;
  c.riemann_kind = riemann_kind;
  const std::vector<R>* stage_in[2] = {&Ustart, &U1};
  for (int st = 0; st < 2; ++st) {
    const std::vector<R>& Uin = *stage_in[st];
    std::vector<Prim<R>> V(c.N);
    for (int64_t i = 0; i < c.N; ++i) V[i] = c.prim_of(Uin.data(), i);
    for (int a = 0; a < D; ++a) {
      const R lambda = (st == 0 ? R(0.5) * dt : dt) / c.dr[a];
      (void)lambda;
      const int64_t na = c.n[a];
      const int64_t stride = a == 0 ? 1 : (a == 1 ? c.n[0] : c.n[0] * c.n[1]);
      const int64_t nlines = c.N / na;
      for (int64_t l = 0; l < nlines; ++l) {
        const int64_t base = a == 0 ? l * c.n[0] : (a == 1 ? (l / c.n[0]) * c.n[0] * c.n[1] + (l % c.n[0]) : l);
        std::vector<Prim<R>> lo(na), hi(na);
        for (int64_t i = 0; i < na; ++i)  // ONE interpolation per cell and axis
          c.interpolate(V[base + c.map_index(i - 1, na) * stride], V[base + i * stride],
                        V[base + c.map_index(i + 1, na) * stride], lo[i], hi[i]);
        std::vector<R> Fl(size_t(na + 1) * NF);
        // periodic: na distinct faces (face -1 is face na-1); outflow: na + 1.  Count na: one face per cell.
        for (int64_t f = 0; f < na; ++f) c.riemann(a, hi[f], lo[c.map_index(f + 1, na)], &Fl[size_t(f + 1) * NF]);
        for (int fz = 0; fz < NF; ++fz) Fl[fz] = Fl[size_t(na) * NF + fz];
        R acc;
        for (int64_t i = 0; i < na; ++i)
          for (int fz = 0; fz < NF; ++fz) {
            const R dF = Fl[size_t(i) * NF + fz] - Fl[size_t(i + 1) * NF + fz];
            acc = std::fma(lambda, dF, acc);
          }
      }
    }
  }
  // CFL term of the new state: prim_of + speed per cell (the kernels form it in the stage-2 epilogue)
  c.U = s.U;
  (void)c.cfl_S();
  store(g_tally, out + NCLASS);
}

}  // namespace

extern "C" int oracle_count_ops(int dims, const int64_t* n, const double* extent, double gamma, int dtype, int boundary,
                                int riemann_kind, const void* U, double cfl, uint64_t* out /* [20] */) {
  if (dtype == 0) {
    if (dims == 1) count<float, 1>(n, extent, gamma, boundary, riemann_kind, (const float*)U, cfl, out);
    else if (dims == 2) count<float, 2>(n, extent, gamma, boundary, riemann_kind, (const float*)U, cfl, out);
    else count<float, 3>(n, extent, gamma, boundary, riemann_kind, (const float*)U, cfl, out);
  } else {
    if (dims == 1) count<double, 1>(n, extent, gamma, boundary, riemann_kind, (const double*)U, cfl, out);
    else if (dims == 2) count<double, 2>(n, extent, gamma, boundary, riemann_kind, (const double*)U, cfl, out);
    else count<double, 3>(n, extent, gamma, boundary, riemann_kind, (const double*)U, cfl, out);
  }
  return 0;
}
