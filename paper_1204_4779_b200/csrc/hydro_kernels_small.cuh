// hydro_kernels_small.cuh — 1-D grids of at most 1024 cells (BASELINE config 0: the 256-cell Sod tube): the WHOLE run in
// one kernel launch.  One block, one thread per cell; the conserved state lives in registers, the primitives of the
// stage input in shared memory; every thread computes the two faces of its cell from the five primitive states around
// it (Eq. 19-22, the "Delayed" arrangement of k_delayed: same device functions, same operation order, bit-equal to the
// oracle); the CFL reduction (a0), the time-step control and the step loop run on the device as in the large-grid path
// (hydro_control.cuh), so `nsteps` steps cost one launch instead of 2 nsteps launches of ~3 us of work each.
#pragma once
#include "hydro_kernels_basic.cuh"

namespace ph {

constexpr int SMALL1D_MAX = 1024;
constexpr long long SMALL1D_MAX_STEPS = 4096;  // steps per launch; the host loops over longer runs

template <class Real, int RS, int LIM>
__global__ void __launch_bounds__(SMALL1D_MAX) k_small1d(Real* U, Geom<Real> g, Scalars* sc, long long nsteps) {
  constexpr int D = 1, NF = 3;
  __shared__ Real Vs[NF][SMALL1D_MAX];
  __shared__ Scalars lsc;  // the handle's scalar block, kept on chip for the whole run and written back at the end
  __shared__ Real s_warp[32];
  __shared__ int s_bad[32];
  const int n = g.n[0], i = threadIdx.x, bnd = g.boundary;
  const bool cell = i < n;
  if (i == 0) lsc = *sc;
  __syncthreads();
  volatile Scalars* vsc = &lsc;
  Real u0[NF] = {Real(1), Real(0), Real(1)};
  if (cell) load_fields_rw<Real, NF>(U, g.N, i, u0);

  // U_out = AddFlux(lam, Flux(U_in), U_base) for this thread's cell (Eq. 19-23)
  auto stage = [&](const Real (&uin)[NF], const Real (&ubase)[NF], Real lam, Real (&uout)[NF]) {
    if (cell) {
      const Prim<Real, D> V = prim_of<Real, D>(uin, g.gm1);
      Vs[0][i] = V.rho;
      Vs[1][i] = V.v[0];
      Vs[2][i] = V.p;
    }
    __syncthreads();
    if (cell) {
      Prim<Real, D> W[5];  // cells i-2 .. i+2 through the boundary's index map
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const int c = map_index(i - 2 + q, n, bnd);
        W[q].rho = Vs[0][c];
        W[q].v[0] = Vs[1][c];
        W[q].p = Vs[2][c];
      }
      Prim<Real, D> hi_m, lo_c, hi_c, lo_p;
      interpolate<Real, D, LIM>(W[0], W[1], W[2], nullptr, &hi_m);
      interpolate<Real, D, LIM>(W[1], W[2], W[3], &lo_c, &hi_c);
      interpolate<Real, D, LIM>(W[2], W[3], W[4], &lo_p, nullptr);
      Real Fm[NF], Fp[NF];
      riemann_flux<Real, D, 0, RS>(g.gamma, g.igm1, hi_m, lo_c, Fm);
      riemann_flux<Real, D, 0, RS>(g.gamma, g.igm1, hi_c, lo_p, Fp);
#pragma unroll
      for (int f = 0; f < NF; ++f) uout[f] = rfma(lam, Fm[f] - Fp[f], ubase[f]);
    }
    __syncthreads();  // every reader of Vs is done before the next stage overwrites it
  };

  for (long long s = 0; s < nsteps; ++s) {
    if (vsc->done) break;  // t_end reached (uniform: every thread reads the same flag after the barrier below)
    const Real lam1 = Real(vsc->lam[0][0]), lam2 = Real(vsc->lam[1][0]);
    Real u1[NF] = {Real(1), Real(0), Real(1)}, u2[NF] = {Real(1), Real(0), Real(1)};
    stage(u0, u0, lam1, u1);
    if (g.integrator == 1) {  // Heun (R20): U2 = 0.5 (U0 + (U1 + dt L(U1)))
      stage(u1, u1, lam2, u2);
#pragma unroll
      for (int f = 0; f < NF; ++f) u2[f] = Real(0.5) * (u0[f] + u2[f]);
    } else {
      stage(u1, u0, lam2, u2);
    }
    Real smax = Real(0);
    int bad = 0;
    if (cell) {
#pragma unroll
      for (int f = 0; f < NF; ++f) u0[f] = u2[f];
      Real ir;
      const Prim<Real, D> V = prim_of<Real, D>(u0, g.gm1, &ir);
      smax = cfl_speed<Real, D>(V, ir, g.gamma, g.idr);
      bad = bad_state<Real, D>(V, u0[NF - 1]);
    }
    // a0 and the time-step control of hydro_control.cuh for ONE block: lanes by butterfly, warps through shared memory,
    // thread 0 finishes the step (S, t, the step counter) and plans the next dt, all in the on-chip copy
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      smax = rmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
      bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((i & 31) == 0) {
      s_warp[i >> 5] = smax;
      s_bad[i >> 5] = bad;
    }
    __syncthreads();
    if (i == 0) {
      Real S = Real(0);
      int nb = 0;
      for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
        S = rmax(S, s_warp[w]);
        nb += s_bad[w];
      }
      lsc.S_last = double(S);
      lsc.nonfinite += nb;
      lsc.t = lsc.last ? lsc.t_end : lsc.t + lsc.dt;
      lsc.steps += 1;
      if (lsc.auto_dt) plan_next_step(&lsc, g);
    }
    __syncthreads();
  }
  if (cell) store_fields<Real, NF>(U, g.N, i, u0);
  if (i == 0) *sc = lsc;
}

}  // namespace ph
