// hydro_kernels_pack.cuh — the fused RK-stage kernel, third design ("pack"): fp32, TWO x-adjacent cells per thread on
// the packed sm_100 instructions FADD2 / FMUL2 / FFMA2, built so that the packed arithmetic fits 128 registers and
// sixteen warps per SM (profiles/r2_README.md: the r1 packed kernel needed 213 registers, two warps per scheduler,
// and lost to the scalar kernel for that reason alone).
//
// Same tile / marching scheme as k_march (hydro_kernels_march.cuh): a block = TY main warps, one row of 64 cells each
// (3-D; in 2-D NWX warps side by side on one row), plus ONE halo warp; the tile is marched through `depth` planes of
// the last axis; every primitive recovery, slope and Riemann solve of a cell / face is done once (Fig. 6-7
// :435-472, "Manifest in SRAM").  What differs:
//   * the rolling window along the marching axis does not live in registers.  The primitives of planes m, m+1, m+2
//     sit in a ring of three shared-memory planes (plane m with its 2-cell star halo); the high-side state of plane m
//     and the flux through face m-1/2 sit in per-thread shared-memory slots.  No register rotates at the loop edge.
//   * x-neighbours exchange by warp shuffle at once (before the barrier); only the y direction and the warp-edge
//     lanes wait for a block barrier.
// Arithmetic: DESIGN.md §4 through the lane-generic functions of hydro_math.cuh with T = f32x2, bit-identical per
// lane to the scalar kernels and to the oracle (tests/test_gpu_parity.py).  n_x must be even (pairs are 8-byte
// aligned and wrap as pairs); the launcher falls back to k_march otherwise.
#pragma once
#include <type_traits>

#include "hydro_kernels_march.cuh"

// fp64, 2-D rows: blocks per SM the register cap of __launch_bounds__ is set for
#ifndef PH_PACK64_MINB2
#define PH_PACK64_MINB2 4
#endif
// fp32, 2-D rows: likewise
#ifndef PH_PACK32_MINB2
#define PH_PACK32_MINB2 2
#endif

namespace ph {

template <class T, int D, int NWX, int TY, int NH = 1>
struct PackShape {
  using S = scalar_t<T>;
  static constexpr int W = LaneTraits<T>::W;             // cells per thread: 2 (f32x2) or 1 (double); 8 bytes either way
  static constexpr int NF = D + 2;
  static constexpr int TXC = NWX * 32 * W;               // cells per tile row
  static constexpr int PX = TXC + 4;                     // plane row: tile + 2 halo cells on each side
  static constexpr int PY = (D == 3) ? TY + 4 : 1;
  static constexpr int OY = (D == 3) ? 2 : 0;
  static constexpr int NMAIN = NWX * TY * 32;
  static constexpr int NT = NMAIN + 32 * NH;               // NH halo warps follow the main warps
  static constexpr int XROWS = (D == 3) ? TY : 1;
  static_assert(D == 2 || D == 3, "2-D and 3-D grids");
  static_assert(NH == 1 || (NH == 2 && D == 3) || (NH == 0 && D == 2),
                "two halo warps (one for the y faces, one for the x faces): 3-D only; no halo warp: 2-D only");
  // NH = 0 (2-D rows): no halo warp.  Neighbouring tiles overlap by 4 cells instead: the first two and the last two cells
  // of a tile row are ghosts that the block loads, converts and reconstructs like its own cells but never stores, so
  // every face of an owned cell lies between two cells of the same block and x needs nothing but the warp shuffles and
  // the warp-edge slots (2 ghost cells per side = the stencil reach).  TXO = owned cells per tile row.
  static constexpr int GH = (NH == 0) ? 2 : 0;
  static constexpr int TXO = TXC - 2 * GH;
  static_assert(D == 3 || TY == 1, "2-D tiles are rows");
  static_assert(D == 2 || NWX == 1, "3-D tiles are one warp wide");
  static_assert((XROWS + W - 1) / W <= 32, "tile too tall for one halo warp");
  struct Smem {
    S V[3][NF][PY][PX];                               // ring: primitives of planes m (with halo), m+1, m+2
    S Hm[NF][XROWS][TXC];                             // high-side marching-axis state of plane m, own cells
    S Fp[NF][XROWS][TXC];                             // flux through the marching-axis face m-1/2, own cells
    S LOy[(D == 3) ? NF : 1][XROWS + 1][(D == 3) ? TXC : 2];  // [r]: low-side y state of tile row r (r = TY: halo warp)
    S Fy[(D == 3) ? NF : 1][XROWS][(D == 3) ? TXC : 2];       // [r]: flux through the low y face of row r (r = 0: halo warp)
    S Un[NF][XROWS][TXC];                             // cp.async staging: U_in of plane m+2, own cells
    S Ub[NF][XROWS][TXC];                             // cp.async staging: U_base of plane m, own cells
    S LOx[NF][XROWS][NWX + 1];                        // [e]: low-side x state of the first cell of warp column e
    S Fx[NF][XROWS][NWX];                             // [e]: flux through the low x face of warp column e
  };
};

// 8-byte asynchronous copy global -> shared of one pair of cells (cp.async: SASS LDGSTS), read back by the issuing
// thread after cp_async_wait_all(): no register is held while the load is in flight
__device__ __forceinline__ void cp_async8(void* dst_smem, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(float* dst_smem, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_addr(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// BND: the boundary mode as a compile-time constant.  On periodic grids (n_x even) every pair of cells a thread
// touches, ghost pairs included, is one aligned 8-byte pair in memory; outflow ghosts are clamped cell by cell.
template <class T, int D, int RS, int STAGE, int NWX, int TY, int MINB, int BND, int NH, int LIM>
__global__ void __launch_bounds__(PackShape<T, D, NWX, TY, NH>::NT, MINB)
    k_pack(const scalar_t<T>* __restrict__ Uin, const scalar_t<T>* Ubase, scalar_t<T>* Uout, Geom<scalar_t<T>> g, Scalars* sc,
           int depth) {
  using Sh = PackShape<T, D, NWX, TY, NH>;
  using S = scalar_t<T>;
  using P = Prim<T, D>;
  constexpr int NF = Sh::NF, TXC = Sh::TXC, OY = Sh::OY, XROWS = Sh::XROWS;
  constexpr int M = D - 1;  // marching axis
  constexpr int W = Sh::W;

  if (sc->done) return;
  extern __shared__ __align__(128) unsigned char pack_smem_raw[];
  typename Sh::Smem& sm = *reinterpret_cast<typename Sh::Smem*>(pack_smem_raw);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nx = g.n[0], ny = g.n[1], nM = g.n[M];
  constexpr int bnd = BND;
  const int x0 = blockIdx.x * Sh::TXO - Sh::GH;  // global x of tile column 0 (NH = 0: a ghost cell)
  const int y0 = (D == 3) ? blockIdx.y * TY : 0;
  const int bm = (D == 3) ? blockIdx.z : blockIdx.y;
  const int m0 = bm * depth;
  const int m1 = min(m0 + depth, nM);
  const int Ni = int(g.N);
  const int psi = (D == 3) ? nx * ny : nx;
  auto plane_of = [&](int m) { return map_index(m, nM, bnd) * psi; };
  auto grid_row = [&](int gj) { return (D == 3) ? march_src(gj, ny, bnd) * nx : 0; };
  // the W cells of a CellSrc: one 8-byte load when they are known to be a pair
  auto ldg_pair = [&](const S* __restrict__ A, int base, const CellSrc& c) {
    if constexpr (W == 2 && BND == BOUNDARY_PERIODIC) return f32x2(__ldg(reinterpret_cast<const float2*>(A + (base + c.o0))));
    else return ldg_cells<T>(A, base, c);
  };

  S s_max = S(0);
  int bad = 0;

  if (warp < NWX * TY) {
    // =========================================================================== main warps
    const int wx = (D == 3) ? 0 : warp;
    const int row = (D == 3) ? warp : 0;
    const int c0 = (wx * 32 + lane) * W;  // first own cell, tile coordinates
    const int gi = x0 + c0;
    const int gj = y0 + row;
    const int pc = c0 + 2, pr = row + OY;
    const bool active = gi < nx && (D == 2 || gj < ny) && c0 >= Sh::GH && c0 < TXC - Sh::GH;
    const CellSrc src = cell_src<T>(gi, grid_row(gj), nx, bnd);
    const int own = (D == 3 ? gj * nx : 0) + gi;

    auto load_cells_of = [&](int m, T (&u)[NF]) {
      const int pl = plane_of(m);
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = ldg_pair(Uin, f * Ni + pl, src);
    };
    // asynchronous copies into this thread's staging slots: U_in of plane mi (own cells) and, when cell >= 0, the
    // own-cell U_base of the plane being updated
    auto stage_copies = [&](int mi, int cell) {
      const int pl = plane_of(mi);
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        if constexpr (W == 1 || BND == BOUNDARY_PERIODIC) {
          cp_async8(&sm.Un[f][row][c0], Uin + (f * Ni + pl + src.o0));
        } else {
          cp_async4(&sm.Un[f][row][c0], Uin + (f * Ni + pl + src.o0));
          cp_async4(&sm.Un[f][row][c0 + 1], Uin + (f * Ni + pl + src.o1));
        }
        if (active && cell >= 0) cp_async8(&sm.Ub[f][row][c0], Ubase + (f * Ni + cell));
      }
    };
    const S lam0 = S(sc->lam[STAGE - 1][0]);
    const S lam1 = S(sc->lam[STAGE - 1][1]);
    const S lam2 = (D == 3) ? S(sc->lam[STAGE - 1][2]) : S(0);

    // ---- prologue: planes m0, m0+1 of the ring, the high-side state of plane m0 and the flux through face m0-1/2
    {
      T u[NF];
      load_cells_of(m0 - 2, u);
      const P Vm2 = prim_of<T, D>(u, g.gm1);
      load_cells_of(m0 - 1, u);
      const P Vm1 = prim_of<T, D>(u, g.gm1);
      load_cells_of(m0, u);
      const P Vc = prim_of<T, D>(u, g.gm1);
      load_cells_of(m0 + 1, u);
      const P Vp1 = prim_of<T, D>(u, g.gm1);
      P him1, loc, hiM;
      interpolate<T, D, LIM>(Vm2, Vm1, Vc, nullptr, &him1);
      interpolate<T, D, LIM>(Vm1, Vc, Vp1, &loc, &hiM);
      T F[NF], a[NF];
      riemann_flux<T, D, M, RS>(g.gamma, g.igm1, him1, loc, F);
      prim_to_fields<T, D>(Vc, a);
#pragma unroll
      for (int f = 0; f < NF; ++f) sts(&sm.V[0][f][pr][pc], a[f]);
      prim_to_fields<T, D>(Vp1, a);
#pragma unroll
      for (int f = 0; f < NF; ++f) sts(&sm.V[1][f][pr][pc], a[f]);
      prim_to_fields<T, D>(hiM, a);
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        sts(&sm.Hm[f][row][c0], a[f]);
        sts(&sm.Fp[f][row][c0], F[f]);
      }
    }
    stage_copies(m0 + 2, -1);
    block_barrier();

    int s0 = 0, s1 = 1, s2 = 2;  // ring slots of planes m, m+1, m+2
    for (int m = m0; m < m1; ++m) {
      // ------------------------------------------------------------ phase A
      const int cell = plane_of(m) + own;
      T vc[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) vc[f] = lds<T>(&sm.V[s0][f][pr][pc]);
      // marching axis: V[m+2] (its U_in was copied during the previous iteration), slope of cell m+1, flux through
      // face m+1/2; then the copies of U_in of plane m+3 (next iteration) and of the own-cell U_base of plane m (phase C)
      T dFm[NF];
      auto z_part = [&]() {
        cp_async_wait_all();
        T un[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) un[f] = lds<T>(&sm.Un[f][row][c0]);
        stage_copies(m + 3, cell);
        const P Vp2 = prim_of<T, D>(un, g.gm1);
        T vp2[NF], loM1[NF], hiM[NF];
        prim_to_fields<T, D>(Vp2, vp2);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          sts(&sm.V[s2][f][pr][pc], vp2[f]);
          const T vp1 = lds<T>(&sm.V[s1][f][pr][pc]);
          const T dy = limited_dy<LIM>(vc[f], vp1, vp2[f]);
          loM1[f] = rfma(S(-0.5), dy, vp1);
          hiM[f] = lds<T>(&sm.Hm[f][row][c0]);
          sts(&sm.Hm[f][row][c0], rfma(S(0.5), dy, vp1));
        }
        T Fn[NF];
        riemann_flux<T, D, M, RS>(g.gamma, g.igm1, prim_from_fields<T, D>(hiM), prim_from_fields<T, D>(loM1), Fn);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          dFm[f] = lds<T>(&sm.Fp[f][row][c0]) - Fn[f];
          sts(&sm.Fp[f][row][c0], Fn[f]);
        }
      };
      // x slopes; the low-side state goes to the left neighbour at once (shuffle), lane 31 is patched after the barrier
      T hix[NF], rs[NF];
      T hiy[(D == 3) ? NF : 1];
      auto xy_slopes = [&]() {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const T l = xshift_left(vc[f], sm.V[s0][f][pr][pc - 1]);
        const T r = xshift_right(vc[f], sm.V[s0][f][pr][pc + W]);
        const T dy = limited_dy<LIM>(l, vc[f], r);
        const T lox = rfma(S(-0.5), dy, vc[f]);
        hix[f] = rfma(S(0.5), dy, vc[f]);
        if (lane == 0) sm.LOx[f][row][wx] = lane_first(lox);
        rs[f] = xshift_right(lox, shfl_dn(lane_first(lox)));
      }
      if constexpr (D == 3) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          const T dy = limited_dy<LIM>(lds<T>(&sm.V[s0][f][pr - 1][pc]), vc[f], lds<T>(&sm.V[s0][f][pr + 1][pc]));
          sts(&sm.LOy[f][row][c0], rfma(S(-0.5), dy, vc[f]));
          hiy[f] = rfma(S(0.5), dy, vc[f]);
        }
      }
      };
      z_part();
      xy_slopes();
      block_barrier();

      // ------------------------------------------------------------ phase B: one Riemann solve per in-plane face
      T Fx[NF], Fy[(D == 3) ? NF : 1];
      if (lane == 31) {
#pragma unroll
        for (int f = 0; f < NF; ++f) lane_set_last(rs[f], sm.LOx[f][row][wx + 1]);
      }
      riemann_flux<T, D, 0, RS>(g.gamma, g.igm1, prim_from_fields<T, D>(hix), prim_from_fields<T, D>(rs), Fx);
      if (NWX > 1 && lane == 31 && wx + 1 < NWX) {
#pragma unroll
        for (int f = 0; f < NF; ++f) sm.Fx[f][row][wx + 1] = lane_last(Fx[f]);
      }
      if constexpr (D == 3) {
        T a[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) a[f] = lds<T>(&sm.LOy[f][row + 1][c0]);
        riemann_flux<T, D, 1, RS>(g.gamma, g.igm1, prim_from_fields<T, D>(hiy), prim_from_fields<T, D>(a), Fy);
        if (row + 1 < TY) {
#pragma unroll
          for (int f = 0; f < NF; ++f) sts(&sm.Fy[f][row + 1][c0], Fy[f]);
        }
      }
      // own-cell base state of Eq. 23 and the x flux of the left neighbour lane: both this thread's / warp's own data,
      // fetched before the barrier so that only the other warps' results are waited for after it
      cp_async_wait_all();
      T ub[NF];
      S nbx[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        ub[f] = lds<T>(&sm.Ub[f][row][c0]);
        nbx[f] = shfl_up(lane_last(Fx[f]));
      }
      block_barrier();

      // ------------------------------------------------------------ phase C: Eq. 23, axes in the order x, y, z
      T lowx[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        S nb = nbx[f];
        if (lane == 0) nb = sm.Fx[f][row][wx];
        lowx[f] = xshift_left(Fx[f], nb);
      }
      if (active) {
        T u[NF];  // own-cell base state of Eq. 23 (copied in phase A; U_base is overwritten in place only below)
#pragma unroll
        for (int f = 0; f < NF; ++f) u[f] = rfma(lam0, lowx[f] - Fx[f], ub[f]);
        if constexpr (D == 3) {
#pragma unroll
          for (int f = 0; f < NF; ++f) u[f] = rfma(lam1, lds<T>(&sm.Fy[f][row][c0]) - Fy[f], u[f]);
#pragma unroll
          for (int f = 0; f < NF; ++f) u[f] = rfma(lam2, dFm[f], u[f]);
        } else {
#pragma unroll
          for (int f = 0; f < NF; ++f) u[f] = rfma(lam1, dFm[f], u[f]);
        }
        if (STAGE == 2 && g.integrator == 1) {  // Heun: U2 = 0.5 (U0 + (U1 + dt L(U1))); U0 still sits in Uout
#pragma unroll
          for (int f = 0; f < NF; ++f) u[f] = S(0.5) * (ld_cells_rw<T>(Uout, f * Ni + cell) + u[f]);
        }
#pragma unroll
        for (int f = 0; f < NF; ++f) st_cells<T>(Uout, f * Ni + cell, u[f]);
        if (STAGE == 2) {
          T ir;
          const P Vn = prim_of<T, D>(u, g.gm1, &ir);
          s_max = rmax(s_max, lane_max(cfl_speed<T, D>(Vn, ir, g.gamma, g.idr)));
          bad += bad_lanes<T, D>(Vn, u[NF - 1]);
        }
      }
      const int t = s0;
      s0 = s1;
      s1 = s2;
      s2 = t;
    }
  } else if constexpr (NH > 0) {
    // =========================================================================== the halo warp
    // Loads the 2-cell star halo of every plane, converts it to primitives (into the ring slot of the NEXT plane) and
    // computes the faces the tile cannot get from its own cells.  NH = 2: the first halo warp serves the y direction
    // (halo rows, the faces below / above the tile), the second the x direction, so that neither has more work per
    // plane than a main warp and the block barriers do not wait for them.
    const int hw = warp - NWX * TY;
    const bool do_y = (D == 3) && (NH == 1 || hw == 0);
    const bool do_x = (NH == 1 || hw == NH - 1);
    constexpr int XHALO = 4 * XROWS / W;                // x halo slots per plane: rows x {2 cells left, 2 cells right} / W
    constexpr int NXP = (XHALO + 31) / 32;
    CellSrc hsrc[NXP];
    int hpy[NXP], hpx[NXP];
    bool hval[NXP];
#pragma unroll
    for (int q = 0; q < NXP; ++q) {
      const int id = lane + 32 * q;
      hval[q] = do_x && id < XHALO;
      const int r = hval[q] ? (W == 2 ? (id >> 1) : (id >> 2)) : 0;
      const int px = (W == 2) ? ((id & 1) ? TXC + 2 : 0) : ((id & 3) < 2 ? (id & 3) : TXC + (id & 3));
      hpy[q] = r + OY;
      hpx[q] = px;
      hsrc[q] = cell_src<T>(x0 + px - 2, grid_row(y0 + r), nx, bnd);
    }
    constexpr int NYP = (D == 3) ? 4 : 0;  // y halo rows
    CellSrc ysrc[NYP > 0 ? NYP : 1];
#pragma unroll
    for (int q = 0; q < NYP; ++q) ysrc[q] = cell_src<T>(x0 + lane * W, grid_row(y0 + (q < 2 ? q : TY + q) - 2), nx, bnd);
    T Uh[NXP][NF], Uyh[NYP > 0 ? NYP : 1][NF];
    auto load_halo = [&](int m) {
      const int pl = plane_of(m);
#pragma unroll
      for (int q = 0; q < NXP; ++q)
        if (hval[q]) {
#pragma unroll
          for (int f = 0; f < NF; ++f) Uh[q][f] = ldg_pair(Uin, f * Ni + pl, hsrc[q]);
        }
      if (do_y) {
#pragma unroll
        for (int q = 0; q < NYP; ++q) {
#pragma unroll
          for (int f = 0; f < NF; ++f) Uyh[q][f] = ldg_pair(Uin, f * Ni + pl, ysrc[q]);
        }
      }
    };
    auto store_halo = [&](int s) {
      T u[NF];
#pragma unroll
      for (int q = 0; q < NXP; ++q)
        if (hval[q]) {
          prim_to_fields<T, D>(prim_of<T, D>(Uh[q], g.gm1), u);
#pragma unroll
          for (int f = 0; f < NF; ++f) sts(&sm.V[s][f][hpy[q]][hpx[q]], u[f]);
        }
      if (do_y) {
#pragma unroll
        for (int q = 0; q < NYP; ++q) {
          prim_to_fields<T, D>(prim_of<T, D>(Uyh[q], g.gm1), u);
#pragma unroll
          for (int f = 0; f < NF; ++f) sts(&sm.V[s][f][q < 2 ? q : TY + q][lane * W + 2], u[f]);
        }
      }
    };
    // x face tasks: lane l handles tile rows ra (first lane of T) and rb (second lane)
    constexpr int XTASK_LANES = (XROWS + W - 1) / W;
    const bool xtask = do_x && lane < XTASK_LANES;
    const int ra = xtask ? lane : 0;
    const int rb = (W == 2) ? min(ra + XTASK_LANES, XROWS - 1) : ra;
    auto plane_x = [&](int s, int qx) {
      T u[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = lane_pack(sm.V[s][f][ra + OY][qx], sm.V[s][f][rb + OY][qx], (T*)nullptr);
      return prim_from_fields<T, D>(u);
    };
    auto plane_y = [&](int s, int py) {
      T u[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = lds<T>(&sm.V[s][f][py][lane * W + 2]);
      return prim_from_fields<T, D>(u);
    };

    load_halo(m0);
    store_halo(0);
    if (m0 + 1 < m1) load_halo(m0 + 1);
    block_barrier();

    int s0 = 0, s1 = 1, s2 = 2;
    for (int m = m0; m < m1; ++m) {
      const bool more = m + 1 < m1;
      // ---- phase A: high-side states of the cells just below the tile, low-side states of those just above;
      //      primitives of the next plane's halo (loaded during the previous phase B)
      P hiYlow, hiXlow;
      if constexpr (D == 3) if (do_y) {
        interpolate<T, D, LIM>(plane_y(s0, 0), plane_y(s0, 1), plane_y(s0, 2), nullptr, &hiYlow);
        P lo;
        interpolate<T, D, LIM>(plane_y(s0, TY + 1), plane_y(s0, TY + 2), plane_y(s0, TY + 3), &lo, nullptr);
        T a[NF];
        prim_to_fields<T, D>(lo, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) sts(&sm.LOy[f][TY][lane * W], a[f]);
      }
      if (xtask) {
        interpolate<T, D, LIM>(plane_x(s0, 0), plane_x(s0, 1), plane_x(s0, 2), nullptr, &hiXlow);
        P lo;
        interpolate<T, D, LIM>(plane_x(s0, TXC + 1), plane_x(s0, TXC + 2), plane_x(s0, TXC + 3), &lo, nullptr);
        T a[NF];
        prim_to_fields<T, D>(lo, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          sm.LOx[f][ra][NWX] = lane_first(a[f]);
          if (W == 2) sm.LOx[f][rb][NWX] = lane_last(a[f]);
        }
      }
      if (more) store_halo(s1);
      block_barrier();
      // ---- phase B: flux through the tile's low faces; loads of the halo of plane m+2
      if constexpr (D == 3) if (do_y) {
        T a[NF], F[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) a[f] = lds<T>(&sm.LOy[f][0][lane * W]);
        riemann_flux<T, D, 1, RS>(g.gamma, g.igm1, hiYlow, prim_from_fields<T, D>(a), F);
#pragma unroll
        for (int f = 0; f < NF; ++f) sts(&sm.Fy[f][0][lane * W], F[f]);
      }
      if (xtask) {
        T a[NF], F[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) a[f] = lane_pack(sm.LOx[f][ra][0], sm.LOx[f][rb][0], (T*)nullptr);
        riemann_flux<T, D, 0, RS>(g.gamma, g.igm1, hiXlow, prim_from_fields<T, D>(a), F);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          sm.Fx[f][ra][0] = lane_first(F[f]);
          if (W == 2) sm.Fx[f][rb][0] = lane_last(F[f]);
        }
      }
      if (m + 2 < m1) load_halo(m + 2);
      block_barrier();
      const int t = s0;
      s0 = s1;
      s1 = s2;
      s2 = t;
    }
  }
  if (STAGE == 2) {
    const unsigned int nblocks = gridDim.x * gridDim.y * gridDim.z;
    block_reduce_and_finalize<S>(s_max, bad, sc, g, nblocks, 1);
  }
}

// ------------------------------------------------------------------------------------------------
// Planes marched per block when the caller gives none.  A block pays a prologue of about two planes' work, and the
// grid runs in waves of `capacity` blocks: the depth (8 .. 128) is the one that wastes least of both, i.e. maximises
// (blocks / (waves * capacity)) * depth / (depth + 2) * waves / (waves + 0.1); the last factor is the measured
// preference for a few waves over exactly one (the tuner tables of configs 2 and 3); ties go to the deeper march.
inline int pack_default_depth(long long tiles_in_plane, int nM, int capacity) {
  int best = nM < 8 ? nM : 8;
  double best_eff = -1.0;
  int last = 0;
  for (int d = nM < 128 ? nM : 128; d >= 8; --d) {  // deepest first: ties go to the deeper march
    const long long zb = (nM + d - 1) / d;  // marching blocks, then the depth that divides the axis evenly among them
    if (zb > 65535) break;                  // the grid dimension that counts them
    const int depth = int((nM + zb - 1) / zb);
    if (depth == last) continue;
    last = depth;
    const long long blocks = tiles_in_plane * zb;
    const long long waves = (blocks + capacity - 1) / capacity;
    const double eff = double(blocks) / double(waves * capacity) * depth / (depth + 2.0) * double(waves) / (double(waves) + 0.1);
    if (eff > best_eff * 1.0001) {
      best_eff = eff;
      best = depth;
    }
  }
  return best;
}

template <class T, int D, int RS, int STAGE, int NWX, int TY, int MINB, int BND, int NH, int LIM = LIMITER_MINBEE>
static bool launch_pack_bnd(const scalar_t<T>* Uin, const scalar_t<T>* Ubase, scalar_t<T>* Uout, const Geom<scalar_t<T>>& g,
                            Scalars* sc, cudaStream_t stream, int depth) {
  using Sh = PackShape<T, D, NWX, TY, NH>;
  auto kern = k_pack<T, D, RS, STAGE, NWX, TY, MINB, BND, NH, LIM>;
  static int capacity[64] = {};  // blocks of this kernel the whole device holds at once (0: not configured yet)
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
  if (!capacity[dev]) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(typename Sh::Smem)) != cudaSuccess)
      return false;
    int per_sm = 0, sms = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, Sh::NT, sizeof(typename Sh::Smem)) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || per_sm < 1 || sms < 1)
      return false;
    capacity[dev] = per_sm * sms;
  }
  constexpr int M = D - 1;
  dim3 grid, block(Sh::NT, 1, 1);
  grid.x = (g.n[0] + Sh::TXO - 1) / Sh::TXO;
  if (depth <= 0)
    depth = pack_default_depth((long long)grid.x * (D == 3 ? (g.n[1] + TY - 1) / TY : 1), g.n[M], capacity[dev]);
  if (D == 3) {
    grid.y = (g.n[1] + TY - 1) / TY;
    grid.z = (g.n[M] + depth - 1) / depth;
    if (grid.y > 65535u || grid.z > 65535u) return false;
  } else {
    grid.y = (g.n[M] + depth - 1) / depth;
    grid.z = 1;
    if (grid.y > 65535u) return false;
  }
  kern<<<grid, block, sizeof(typename Sh::Smem), stream>>>(Uin, Ubase, Uout, g, sc, depth);
  return true;
}

template <class T, int D, int RS, int STAGE, int NWX, int TY, int MINB, int NH = 1, int LIM = LIMITER_MINBEE>
static bool launch_pack_shape(const scalar_t<T>* Uin, const scalar_t<T>* Ubase, scalar_t<T>* Uout, const Geom<scalar_t<T>>& g,
                              Scalars* sc, cudaStream_t stream, int depth) {
  if (g.boundary == BOUNDARY_PERIODIC)
    return launch_pack_bnd<T, D, RS, STAGE, NWX, TY, MINB, BOUNDARY_PERIODIC, NH, LIM>(Uin, Ubase, Uout, g, sc, stream, depth);
  return launch_pack_bnd<T, D, RS, STAGE, NWX, TY, MINB, BOUNDARY_OUTFLOW, NH, LIM>(Uin, Ubase, Uout, g, sc, stream, depth);
}

// Returns false when the packed kernel does not cover this shape (fp32: odd n_x; unknown block shape): the caller falls back.
//   block[0] (2-D): main warps per block (0 = default); block[1] (3-D): main warps TY (0 = default; 14 = two halo warps)
// Real = float: T = f32x2 (two cells per thread); Real = double: T = double (one cell per thread, same 8 bytes).
template <class Real, int D, int RS, int STAGE>
bool launch_pack_stage(const Real* Uin, const Real* Ubase, Real* Uout, const Geom<Real>& g, Scalars* sc, cudaStream_t stream,
                       const int* block, int tile_depth) {
  if constexpr (D == 1) {
    return false;
  } else {
    constexpr bool F32 = sizeof(Real) == 4;
    using T = typename std::conditional<F32, f32x2, double>::type;
    constexpr int W = LaneTraits<T>::W;
    if (W == 2 && g.n[0] % 2 != 0) return false;
    // a block_* knob this dimension does not read must be 0: "shape not covered", not a silently ignored request
    if (D == 2 ? (block[1] != 0 || block[2] < 0 || block[2] > 1) : (block[0] != 0 || block[2] != 0)) return false;
    if constexpr (D == 2) {
      // 2-D rows: overlapping tiles, no halo warp (block[2] = 1: the halo-warp form of the same kernel).  Default
      // row width: the one of 2 / 4 / 8 warps that leaves the fewest idle lanes (ghost cells + ragged last tile)
      const bool halo_warp = block[2] == 1;
      int nwx = block[0];
      if (nwx <= 0) {
        double best = -1.0;
        for (int c : {2, 4, 8}) {
          const int owned = c * 32 * W - 4;
          // lanes at work; wider rows pay more for their block barriers (measured: 2 warps beat 4 at equal lane use)
          const double eff = double(g.n[0]) / double((long long)((g.n[0] + owned - 1) / owned) * c * 32 * W) *
                             (c == 2 ? 1.0 : (c == 4 ? 0.97 : 0.94));
          if (eff > best * 1.0001) {
            best = eff;
            nwx = c;
          }
        }
        if (halo_warp) nwx = 4;
      }
      const int depth = tile_depth;  // 0: launch_pack_bnd picks it from the kernel's occupancy
      constexpr int MB = F32 ? PH_PACK32_MINB2 : PH_PACK64_MINB2;
      if (!halo_warp) {
        if constexpr (F32)
          if (nwx == 1) return launch_pack_shape<T, D, RS, STAGE, 1, 1, MB, 0>(Uin, Ubase, Uout, g, sc, stream, depth);
        if (nwx == 2) return launch_pack_shape<T, D, RS, STAGE, 2, 1, MB, 0>(Uin, Ubase, Uout, g, sc, stream, depth);
        if (nwx == 4) return launch_pack_shape<T, D, RS, STAGE, 4, 1, MB, 0>(Uin, Ubase, Uout, g, sc, stream, depth);
        if (nwx == 8) return launch_pack_shape<T, D, RS, STAGE, 8, 1, MB, 0>(Uin, Ubase, Uout, g, sc, stream, depth);
        return false;
      }
      if (nwx == 2) return launch_pack_shape<T, D, RS, STAGE, 2, 1, MB>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (nwx == 4) return launch_pack_shape<T, D, RS, STAGE, 4, 1, MB>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (nwx == 7) return launch_pack_shape<T, D, RS, STAGE, 7, 1, MB>(Uin, Ubase, Uout, g, sc, stream, depth);
      return false;
    } else {
      // default tile height: 14 rows + two halo warps (one block of 16 warps per SM: the halo work per cell halves and
      // neither halo warp has more work per plane than a main warp) when the grid gives every SM several such blocks
      // at the full marching depth; 7 rows + one halo warp (two blocks per SM) otherwise (profiles/r2_README.md)
      int ty = block[1];
      const int tw = 32 * W;
      if (ty <= 0) {
        const long long tiles14 = (long long)((g.n[0] + tw - 1) / tw) * ((g.n[1] + 13) / 14);
        ty = tiles14 * ((g.n[2] + 127) / 128) >= 4 * device_sm_count() ? 14 : 7;
      }
      const int depth = tile_depth;  // 0: launch_pack_bnd picks it from the kernel's occupancy
      if (ty == 7) return launch_pack_shape<T, D, RS, STAGE, 1, 7, 2>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (ty == 14) return launch_pack_shape<T, D, RS, STAGE, 1, 14, 1, 2>(Uin, Ubase, Uout, g, sc, stream, depth);
      if constexpr (F32) {
        if (ty == 5) return launch_pack_shape<T, D, RS, STAGE, 1, 5, 2>(Uin, Ubase, Uout, g, sc, stream, depth);
        if (ty == 11) return launch_pack_shape<T, D, RS, STAGE, 1, 11, 1>(Uin, Ubase, Uout, g, sc, stream, depth);
        if (ty == 15) return launch_pack_shape<T, D, RS, STAGE, 1, 15, 1>(Uin, Ubase, Uout, g, sc, stream, depth);
      }
      return false;
    }
  }
}

// The interpolation variants other than MINBEE (LIM = LIMITER_NONE, LIMITER_MC; R22) exist in the default launch
// shapes only (2-D: rows of 2 warps as overlapping tiles; 3-D: 7-row tiles with one halo warp); instantiated in
// pack_lim_f<32|64>_d<D>.cu.
template <class Real, int D, int RS, int STAGE, int LIM>
bool launch_pack_stage_lim(const Real* Uin, const Real* Ubase, Real* Uout, const Geom<Real>& g, Scalars* sc,
                           cudaStream_t stream) {
  if constexpr (D == 1) {
    return false;
  } else {
    constexpr bool F32 = sizeof(Real) == 4;
    using T = typename std::conditional<F32, f32x2, double>::type;
    if (LaneTraits<T>::W == 2 && g.n[0] % 2 != 0) return false;
    if constexpr (D == 2)
      return launch_pack_shape<T, D, RS, STAGE, 2, 1, (F32 ? 2 : PH_PACK64_MINB2), 0, LIM>(Uin, Ubase, Uout, g, sc, stream, 0);
    else
      return launch_pack_shape<T, D, RS, STAGE, 1, 7, 2, 1, LIM>(Uin, Ubase, Uout, g, sc, stream, 0);
  }
}

}  // namespace ph
