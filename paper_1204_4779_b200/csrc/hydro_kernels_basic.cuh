// hydro_kernels_basic.cuh — the Manifest end and the pure Delayed end of the paper's trade-off
// (Fig. 6-7 :435-472, Table 5 :754-770), one thread per cell, no shared memory:
//
//   manifest_all  : k_prim -> k_recon<A> -> k_riemann<A> -> k_update   (V, VL/VR, F_a all in HBM;
//                   the paper's "Hayaakitsuhime": interpolation and Riemann results both Manifest)
//   manifest_flux : k_flux<A> -> k_update                              (only F_a in HBM; the paper's
//                   hand-tuned winner "Shinatsuhiko": Riemann Manifest, interpolation Delayed)
//   delayed       : k_delayed                                          (everything recomputed from U by
//                   every thread; the paper's "Izanami")
//   k_cfl         : standalone CFL reduction (after set_state)
//
// The fused, shared-memory / register-marching kernels live in hydro_kernels_fused.cuh.
#pragma once
#include "hydro_control.cuh"

namespace ph {

template <int D>
__device__ __forceinline__ void decode_cell(long long c, const int (&n)[3], int (&idx)[3]) {
  if (D == 1) {
    idx[0] = int(c);
    idx[1] = idx[2] = 0;
  } else if (D == 2) {
    idx[1] = int(c / n[0]);
    idx[0] = int(c - (long long)idx[1] * n[0]);
    idx[2] = 0;
  } else {
    const long long plane = (long long)n[0] * n[1];
    idx[2] = int(c / plane);
    const long long r = c - idx[2] * plane;
    idx[1] = int(r / n[0]);
    idx[0] = int(r - (long long)idx[1] * n[0]);
  }
}

template <int A>
__device__ __forceinline__ long long axis_stride(const int (&n)[3]) {
  return A == 0 ? 1ll : (A == 1 ? (long long)n[0] : (long long)n[0] * n[1]);
}

// index of the grid line through a cell along axis A (the cell index with i_A removed)
template <int A>
__device__ __forceinline__ long long line_index(const int (&idx)[3], const int (&n)[3]) {
  if (A == 0) return (long long)idx[2] * n[1] + idx[1];
  if (A == 1) return (long long)idx[2] * n[0] + idx[0];
  return (long long)idx[1] * n[0] + idx[0];
}

template <class Real, int NF>
__device__ __forceinline__ void load_fields(const Real* __restrict__ A, long long N, long long c, Real (&u)[NF]) {
#pragma unroll
  for (int f = 0; f < NF; ++f) u[f] = __ldg(A + (size_t)f * N + c);
}
// coherent loads: for U_base, which the last stage overwrites in place (each thread reads only its own cell)
template <class Real, int NF>
__device__ __forceinline__ void load_fields_rw(const Real* A, long long N, long long c, Real (&u)[NF]) {
#pragma unroll
  for (int f = 0; f < NF; ++f) u[f] = A[(size_t)f * N + c];
}
template <class Real, int NF>
__device__ __forceinline__ void store_fields(Real* __restrict__ A, long long N, long long c, const Real (&u)[NF]) {
#pragma unroll
  for (int f = 0; f < NF; ++f) A[(size_t)f * N + c] = u[f];
}
template <class Real, int D>
__device__ __forceinline__ Prim<Real, D> load_prim(const Real* __restrict__ V, long long N, long long c) {
  Real u[D + 2];
  load_fields<Real, D + 2>(V, N, c, u);
  Prim<Real, D> P;
  P.rho = u[0];
#pragma unroll
  for (int b = 0; b < D; ++b) P.v[b] = u[1 + b];
  P.p = u[D + 1];
  return P;
}
template <class Real, int D>
__device__ __forceinline__ void store_prim(Real* __restrict__ V, long long N, long long c, const Prim<Real, D>& P) {
  Real u[D + 2];
  u[0] = P.rho;
#pragma unroll
  for (int b = 0; b < D; ++b) u[1 + b] = P.v[b];
  u[D + 1] = P.p;
  store_fields<Real, D + 2>(V, N, c, u);
}

// flags a cell whose new state is unusable (R19)
template <class Real, int D>
__device__ __forceinline__ int bad_state(const Prim<Real, D>& V, Real E) {
  return !(V.rho > Real(0)) || !(V.p > Real(0)) || !(rabs(E) <= Real(3.0e38));
}

// ------------------------------------------------------------------ standalone CFL reduction (a0)
template <class Real, int D>
__global__ void __launch_bounds__(256) k_cfl(const Real* __restrict__ U, Geom<Real> g, Scalars* sc) {
  Real s = Real(0);
  int bad = 0;
  for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < g.N; c += (long long)gridDim.x * blockDim.x) {
    Real u[D + 2], ir;
    load_fields<Real, D + 2>(U, g.N, c, u);
    const Prim<Real, D> V = prim_of<Real, D>(u, g.gm1, &ir);
    s = rmax(s, cfl_speed<Real, D>(V, ir, g.gamma, g.idr));
    bad += bad_state<Real, D>(V, u[D + 1]);
  }
  block_reduce_and_finalize<Real>(s, bad, sc, g, gridDim.x, 0);
}

// ------------------------------------------------------------------ state_kind = primitive: conversions at the boundary
// TO_CONS: V = (rho, v_a, p) -> U = (rho, rho v_a, E), E = fma(0.5 rho, q, p/(gamma-1)) (EOS PAPER.md:694, DESIGN.md §4
// "cons"); otherwise U -> V by Eq. 19.  in == out is allowed (each thread touches only its own cell).
template <class Real, int D, bool TO_CONS>
__global__ void __launch_bounds__(256) k_convert(const Real* in, Real* out, Geom<Real> g) {
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= g.N) return;
  Real a[D + 2], b[D + 2];
  load_fields_rw<Real, D + 2>(in, g.N, c, a);
  if (TO_CONS) {
    Real q = a[1] * a[1];
#pragma unroll
    for (int d = 1; d < D; ++d) q = rfma(a[1 + d], a[1 + d], q);
    b[0] = a[0];
#pragma unroll
    for (int d = 0; d < D; ++d) b[1 + d] = a[0] * a[1 + d];
    b[D + 1] = rfma(Real(0.5) * a[0], q, a[D + 1] * g.igm1);
  } else {
    const Prim<Real, D> V = prim_of<Real, D>(a, g.gm1);
    b[0] = V.rho;
#pragma unroll
    for (int d = 0; d < D; ++d) b[1 + d] = V.v[d];
    b[D + 1] = V.p;
  }
  store_fields<Real, D + 2>(out, g.N, c, b);
}

// ------------------------------------------------------------------ manifest_all pieces
// a1: V = V(U), Eq. 19
template <class Real, int D>
__global__ void __launch_bounds__(256) k_prim(const Real* __restrict__ U, Real* __restrict__ V, Geom<Real> g,
                                               const Scalars* sc) {
  if (sc->done) return;
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= g.N) return;
  Real u[D + 2];
  load_fields<Real, D + 2>(U, g.N, c, u);
  store_prim<Real, D>(V, g.N, c, prim_of<Real, D>(u, g.gm1));
}

// a2: (VR[i-1/2], VL[i+1/2]) = Interpolate(V[i-1], V[i], V[i+1]) along axis A, Eq. 20-21
template <class Real, int D, int A>
__global__ void __launch_bounds__(256) k_recon(const Real* __restrict__ V, Real* __restrict__ LO, Real* __restrict__ HI,
                                                Geom<Real> g, const Scalars* sc) {
  if (sc->done) return;
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= g.N) return;
  int idx[3];
  decode_cell<D>(c, g.n, idx);
  const long long st = axis_stride<A>(g.n);
  const long long cm = c + (long long)(map_index(idx[A] - 1, g.n[A], g.boundary) - idx[A]) * st;
  const long long cp = c + (long long)(map_index(idx[A] + 1, g.n[A], g.boundary) - idx[A]) * st;
  Prim<Real, D> lo, hi;
  interpolate<Real, D>(load_prim<Real, D>(V, g.N, cm), load_prim<Real, D>(V, g.N, c), load_prim<Real, D>(V, g.N, cp),
                       &lo, &hi);
  store_prim<Real, D>(LO, g.N, c, lo);
  store_prim<Real, D>(HI, g.N, c, hi);
}

// a3: F_A[i+1/2] = Riemann_A(VL[i+1/2], VR[i+1/2]), Eq. 22.  F[c] holds the face on the +A side of cell c;
// with outflow boundaries the thread of i_A = 0 also writes the face on its -A side to Fb[line].
template <class Real, int D, int A, int RS>
__global__ void __launch_bounds__(256) k_riemann(const Real* __restrict__ LO, const Real* __restrict__ HI,
                                                  Real* __restrict__ F, Real* __restrict__ Fb, Geom<Real> g,
                                                  const Scalars* sc) {
  if (sc->done) return;
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= g.N) return;
  int idx[3];
  decode_cell<D>(c, g.n, idx);
  const long long st = axis_stride<A>(g.n);
  const long long cp = c + (long long)(map_index(idx[A] + 1, g.n[A], g.boundary) - idx[A]) * st;
  Real Fl[D + 2];
  riemann_flux<Real, D, A, RS>(g.gamma, g.igm1, load_prim<Real, D>(HI, g.N, c), load_prim<Real, D>(LO, g.N, cp), Fl);
  store_fields<Real, D + 2>(F, g.N, c, Fl);
  if (g.boundary == BOUNDARY_OUTFLOW && idx[A] == 0) {
    // ghost cell -1 is a copy of cell 0 with zero slope: VL = hi(cell 0) = V[0], VR = lo(cell 0) = V[0]
    riemann_flux<Real, D, A, RS>(g.gamma, g.igm1, load_prim<Real, D>(HI, g.N, c), load_prim<Real, D>(LO, g.N, c), Fl);
    store_fields<Real, D + 2>(Fb, g.N / g.n[A], line_index<A>(idx, g.n), Fl);
  }
}

// ------------------------------------------------------------------ flux of one face straight from U
// Face between cells f and f+1 (indices along axis A, mapped through the boundary) on the grid line through
// cell c (whose index along A is iA): prim x4, interpolate x2, riemann (Eq. 19-22).
template <class Real, int D, int A, int RS, int LIM = LIMITER_MINBEE>
__device__ __forceinline__ void face_flux_from_U(const Real* __restrict__ U, const Geom<Real>& g, long long c, int iA,
                                                 int f, Real (&F)[D + 2]) {
  const long long st = axis_stride<A>(g.n);
  Prim<Real, D> V[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const long long cc = c + (long long)(map_index(f - 1 + q, g.n[A], g.boundary) - iA) * st;
    Real u[D + 2];
    load_fields<Real, D + 2>(U, g.N, cc, u);
    V[q] = prim_of<Real, D>(u, g.gm1);
  }
  Prim<Real, D> hi0, lo1;
  interpolate<Real, D, LIM>(V[0], V[1], V[2], nullptr, &hi0);
  interpolate<Real, D, LIM>(V[1], V[2], V[3], &lo1, nullptr);
  riemann_flux<Real, D, A, RS>(g.gamma, g.igm1, hi0, lo1, F);
}

// manifest_flux: a1+a2+a3 fused per axis, F_A to HBM
template <class Real, int D, int A, int RS>
__global__ void __launch_bounds__(256) k_flux(const Real* __restrict__ U, Real* __restrict__ F, Real* __restrict__ Fb,
                                               Geom<Real> g, const Scalars* sc) {
  if (sc->done) return;
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= g.N) return;
  int idx[3];
  decode_cell<D>(c, g.n, idx);
  Real Fl[D + 2];
  face_flux_from_U<Real, D, A, RS>(U, g, c, idx[A], idx[A], Fl);
  store_fields<Real, D + 2>(F, g.N, c, Fl);
  if (g.boundary == BOUNDARY_OUTFLOW && idx[A] == 0) {
    face_flux_from_U<Real, D, A, RS>(U, g, c, idx[A], -1, Fl);
    store_fields<Real, D + 2>(Fb, g.N / g.n[A], line_index<A>(idx, g.n), Fl);
  }
}

template <class Real, int D>
struct FluxArrays {
  const Real* F[3];   // F[a][f*N + c]: face on the +a side of cell c
  const Real* Fb[3];  // outflow only: face on the -a side of the cells with i_a = 0
};

template <class Real, int D, int A>
__device__ __forceinline__ void add_axis(Real (&u)[D + 2], const FluxArrays<Real, D>& fa, const Geom<Real>& g,
                                         long long c, const int (&idx)[3], Real lam) {
  const long long st = axis_stride<A>(g.n);
  Real Fm[D + 2], Fp[D + 2];
  load_fields<Real, D + 2>(fa.F[A], g.N, c, Fp);
  if (g.boundary == BOUNDARY_OUTFLOW && idx[A] == 0)
    load_fields<Real, D + 2>(fa.Fb[A], g.N / g.n[A], line_index<A>(idx, g.n), Fm);
  else
    load_fields<Real, D + 2>(fa.F[A], g.N, c + (long long)(map_index(idx[A] - 1, g.n[A], g.boundary) - idx[A]) * st, Fm);
#pragma unroll
  for (int f = 0; f < D + 2; ++f) u[f] = rfma(lam, Fm[f] - Fp[f], u[f]);
}

// a4 (+ a0 in the last stage): U_out = U_base + sum_a lambda_a (F_a[i-1/2] - F_a[i+1/2]), Eq. 23
template <class Real, int D, int STAGE>
__global__ void __launch_bounds__(256) k_update(const Real* Ubase, Real* Uout,
                                                 FluxArrays<Real, D> fa, Geom<Real> g, Scalars* sc) {
  if (sc->done) return;
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  Real s = Real(0);
  int bad = 0;
  if (c < g.N) {
    int idx[3];
    decode_cell<D>(c, g.n, idx);
    Real u[D + 2];
    load_fields_rw<Real, D + 2>(Ubase, g.N, c, u);
    add_axis<Real, D, 0>(u, fa, g, c, idx, Real(sc->lam[STAGE - 1][0]));
    if constexpr (D > 1) add_axis<Real, D, 1>(u, fa, g, c, idx, Real(sc->lam[STAGE - 1][1]));
    if constexpr (D > 2) add_axis<Real, D, 2>(u, fa, g, c, idx, Real(sc->lam[STAGE - 1][2]));
    if (STAGE == 2 && g.integrator == 1) {  // Heun: U2 = 0.5 (U0 + (U1 + dt L(U1))); U0 still sits in Uout
      Real u0[D + 2];
      load_fields_rw<Real, D + 2>(Uout, g.N, c, u0);
#pragma unroll
      for (int f = 0; f < D + 2; ++f) u[f] = Real(0.5) * (u0[f] + u[f]);
    }
    store_fields<Real, D + 2>(Uout, g.N, c, u);
    if (STAGE == 2) {
      Real ir;
      const Prim<Real, D> V = prim_of<Real, D>(u, g.gm1, &ir);
      s = cfl_speed<Real, D>(V, ir, g.gamma, g.idr);
      bad = bad_state<Real, D>(V, u[D + 1]);
    }
  }
  if (STAGE == 2) block_reduce_and_finalize<Real>(s, bad, sc, g, gridDim.x, 1);
}

// ------------------------------------------------------------------ prescribed ghost cells (R23)
// The outermost two cells of every axis := G's (the analytic solution is substituted into the ghost
// cells).  One thread per cell; the cells in between are left alone.
template <class Real, int D>
__global__ void __launch_bounds__(256) k_inject_ghosts(Real* __restrict__ U, const Real* __restrict__ G, Geom<Real> g) {
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= g.N) return;
  int idx[3];
  decode_cell<D>(c, g.n, idx);
  bool ghost = false;
#pragma unroll
  for (int a = 0; a < D; ++a) ghost = ghost || idx[a] < 2 || idx[a] >= g.n[a] - 2;
  if (!ghost) return;
#pragma unroll
  for (int f = 0; f < D + 2; ++f) U[(size_t)f * g.N + c] = G[(size_t)f * g.N + c];
}

// ------------------------------------------------------------------ delayed: one kernel per stage, no sharing
template <class Real, int D, int A, int RS, int LIM>
__device__ __forceinline__ void delayed_axis(Real (&u)[D + 2], const Real* __restrict__ Uin, const Geom<Real>& g,
                                             long long c, const int (&idx)[3], Real lam) {
  Real Fm[D + 2], Fp[D + 2];
  face_flux_from_U<Real, D, A, RS, LIM>(Uin, g, c, idx[A], idx[A] - 1, Fm);
  face_flux_from_U<Real, D, A, RS, LIM>(Uin, g, c, idx[A], idx[A], Fp);
#pragma unroll
  for (int f = 0; f < D + 2; ++f) u[f] = rfma(lam, Fm[f] - Fp[f], u[f]);
}

// LIM: the interpolation variant (R22), a compile-time parameter like the Riemann solver
template <class Real, int D, int RS, int STAGE, int LIM = LIMITER_MINBEE>
__global__ void __launch_bounds__(128) k_delayed(const Real* __restrict__ Uin, const Real* Ubase, Real* Uout,
                                                  Geom<Real> g, Scalars* sc) {
  if (sc->done) return;
  const long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  Real s = Real(0);
  int bad = 0;
  if (c < g.N) {
    int idx[3];
    decode_cell<D>(c, g.n, idx);
    Real u[D + 2];
    load_fields_rw<Real, D + 2>(Ubase, g.N, c, u);
    delayed_axis<Real, D, 0, RS, LIM>(u, Uin, g, c, idx, Real(sc->lam[STAGE - 1][0]));
    if constexpr (D > 1) delayed_axis<Real, D, 1, RS, LIM>(u, Uin, g, c, idx, Real(sc->lam[STAGE - 1][1]));
    if constexpr (D > 2) delayed_axis<Real, D, 2, RS, LIM>(u, Uin, g, c, idx, Real(sc->lam[STAGE - 1][2]));
    if (STAGE == 2 && g.integrator == 1) {  // Heun: U2 = 0.5 (U0 + (U1 + dt L(U1))); U0 still sits in Uout
      Real u0[D + 2];
      load_fields_rw<Real, D + 2>(Uout, g.N, c, u0);
#pragma unroll
      for (int f = 0; f < D + 2; ++f) u[f] = Real(0.5) * (u0[f] + u[f]);
    }
    store_fields<Real, D + 2>(Uout, g.N, c, u);
    if (STAGE == 2) {
      Real ir;
      const Prim<Real, D> V = prim_of<Real, D>(u, g.gm1, &ir);
      s = cfl_speed<Real, D>(V, ir, g.gamma, g.idr);
      bad = bad_state<Real, D>(V, u[D + 1]);
    }
  }
  if (STAGE == 2) block_reduce_and_finalize<Real>(s, bad, sc, g, gridDim.x, 1);
}

}  // namespace ph
