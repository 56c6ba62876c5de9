// hydro_kernels_fused.cuh — the fused end of the Manifest <-> Delayed axis: ONE kernel per RK stage,
// every intermediate (primitives, interface states, fluxes) kept on chip and computed exactly once
// per cell / face ("Manifest in SRAM"), Fig. 6-7 :435-472 rebuilt for sm_100a.
//
// Decomposition (D = 2, 3; 1-D grids use k_delayed):
//   * a block owns a TX x TY tile of the plane spanned by the leading axes (x for D = 2, x-y for D = 3)
//     and MARCHES along the last axis M (y for D = 2, z for D = 3) through `depth` planes;
//   * along M every thread keeps a rolling register window of its own column: V[m], V[m+1], V[m+2],
//     the +M interface state of cell m and the flux through the face m-1/2, so each primitive
//     recovery (Eq. 19), each MINBEE slope (Eq. 20-21) and each Riemann solve (Eq. 22) along M is
//     done once;
//   * inside the plane the primitives of the tile plus a 2-cell star halo sit in shared memory
//     (double-buffered over planes); every thread reconstructs its own cell once per axis, hands the
//     low-side interface state to its lower neighbour and the face flux to its upper neighbour
//     through one shared-memory exchange slot per cell and axis (lo first, then F, same slot);
//   * the two things a tile cannot get from its own threads — the lo state of the first cell beyond
//     the tile and the flux through the tile's lowest face — are produced by TX + TY "halo tasks"
//     batched into at most two warps;
//   * Eq. 23 is applied in the order x, y, z onto U_base (R11); the last stage forms the
//     primitives of the new state in registers and feeds the CFL max (a0) into the block reduction.
// Ragged tiles and periodic / outflow ghosts need no special cases: a plane position with global index
// g outside [0, n) simply holds the state of cell map_index(min(g, n + 1)), loaded by whichever thread
// owns that position; threads whose own cell lies outside the grid compute but never store.
#pragma once
#include "hydro_kernels_basic.cuh"

namespace ph {

template <class Real, int D, int TX, int TY>
struct FusedSmem {
  static constexpr int NF = D + 2;
  static constexpr int PX = TX + 4;
  static constexpr int PY = (D == 3) ? TY + 4 : 1;
  static constexpr int OY = (D == 3) ? 2 : 0;  // row of the tile's first cell inside the padded plane
  Real V[2][NF][PY][PX];                       // primitives of plane m (buffer m & 1 ... toggled), halo 2
  Real Ex[NF][TY][TX + 1];                     // x exchange: slot i = lo of cell i, then F through face i-1/2
  Real Ey[(D == 3) ? NF : 1][(D == 3) ? TY + 1 : 1][(D == 3) ? TX : 1];
};

// global index of the cell whose state plane position g (>= -2) holds
__device__ __forceinline__ int src_index(int g, int n, int boundary) {
  return map_index(g > n + 1 ? n + 1 : g, n, boundary);
}

template <class Real, int D>
__device__ __forceinline__ Prim<Real, D> prim_from_array(const Real (&u)[D + 2]) {
  Prim<Real, D> P;
  P.rho = u[0];
#pragma unroll
  for (int b = 0; b < D; ++b) P.v[b] = u[1 + b];
  P.p = u[D + 1];
  return P;
}
template <class Real, int D>
__device__ __forceinline__ void prim_to_array(const Prim<Real, D>& P, Real (&u)[D + 2]) {
  u[0] = P.rho;
#pragma unroll
  for (int b = 0; b < D; ++b) u[1 + b] = P.v[b];
  u[D + 1] = P.p;
}

template <class Real, int D, int RS, int STAGE, int TX, int TY>
__global__ void __launch_bounds__(TX* TY)
    k_fused(const Real* __restrict__ Uin, const Real* Ubase, Real* Uout, Geom<Real> g, Scalars* sc, int depth) {
  static_assert(D == 2 || D == 3, "the marching kernel covers 2-D and 3-D grids");
  static_assert(D == 3 || TY == 1, "2-D tiles are rows");
  static_assert(TX % 32 == 0 && TY <= 32, "tile shape");
  using Smem = FusedSmem<Real, D, TX, TY>;
  using P = Prim<Real, D>;
  constexpr int NF = D + 2;
  constexpr int M = D - 1;  // marching axis
  constexpr int NT = TX * TY;
  constexpr int OY = Smem::OY;
  constexpr int HX = 4 * TY;                          // halo cells beside the tile along x
  constexpr int H = HX + (D == 3 ? 4 * TX : 0);       // ... plus below / above it along y
  constexpr int YTASK0 = NT - TX;                     // D = 3: threads [YTASK0, NT) run the y halo tasks
  constexpr int XTASK0 = (D == 3) ? NT - TX - 32 : NT - 1;  // threads [XTASK0, XTASK0 + TY) run the x halo tasks
  static_assert(H <= NT && XTASK0 >= 0, "tile too small for its halo work");

  if (sc->done) return;
  extern __shared__ __align__(16) unsigned char fused_smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(fused_smem_raw);

  const int li = threadIdx.x;
  const int lj = (D == 3) ? threadIdx.y : 0;
  const int t = lj * TX + li;
  const int x0 = blockIdx.x * TX;
  const int y0 = (D == 3) ? blockIdx.y * TY : 0;
  const int bm = (D == 3) ? blockIdx.z : blockIdx.y;
  const int nM = g.n[M];
  const int m0 = bm * depth;
  const int m1 = min(m0 + depth, nM);
  const int bnd = g.boundary;
  const int gi = x0 + li, gj = y0 + lj;
  const bool active = gi < g.n[0] && (D == 2 || gj < g.n[1]);
  const long long N = g.N;
  const long long ps = (D == 3) ? (long long)g.n[0] * g.n[1] : (long long)g.n[0];
  const long long col = (D == 3 ? (long long)src_index(gj, g.n[1], bnd) * g.n[0] : 0ll) + src_index(gi, g.n[0], bnd);
  const long long own = (D == 3 ? (long long)gj * g.n[0] : 0ll) + gi;  // valid when active

  // halo cells of the plane: one per thread t < H
  const bool is_halo = t < H;
  int hpx = 0, hpy = 0;
  long long hcol = 0;
  if (is_halo) {
    if (t < HX) {
      const int r = t >> 2, q = t & 3;
      hpx = q < 2 ? q - 2 : TX + q - 2;
      hpy = r;
    } else {
      const int u = t - HX;
      const int q = u / TX;
      hpx = u - q * TX;
      hpy = q < 2 ? q - 2 : TY + q - 2;
    }
    hcol = (D == 3 ? (long long)src_index(y0 + hpy, g.n[1], bnd) * g.n[0] : 0ll) + src_index(x0 + hpx, g.n[0], bnd);
  }

  auto plane_of = [&](int m) { return (long long)map_index(m, nM, bnd) * ps; };
  auto load_prim_at = [&](long long c) {
    Real u[NF];
    load_fields<Real, NF>(Uin, N, c, u);
    return prim_of<Real, D>(u, g.gm1);
  };
  auto sts_plane = [&](int b, int py, int px, const P& V) {
    Real u[NF];
    prim_to_array<Real, D>(V, u);
#pragma unroll
    for (int f = 0; f < NF; ++f) sm.V[b][f][py][px] = u[f];
  };
  auto lds_plane = [&](int b, int py, int px) {
    Real u[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) u[f] = sm.V[b][f][py][px];
    return prim_from_array<Real, D>(u);
  };

  const Real lam0 = Real(sc->lam[STAGE - 1][0]);
  const Real lam1 = Real(sc->lam[STAGE - 1][1]);
  const Real lam2 = (D == 3) ? Real(sc->lam[STAGE - 1][2]) : Real(0);

  // ---------------------------------------------------------------- prologue: window at m0
  P Vc, Vp1, hiM;
  Real Fprev[NF], Unext[NF], Uh[NF];
  {
    const P Vm2 = load_prim_at(plane_of(m0 - 2) + col);
    const P Vm1 = load_prim_at(plane_of(m0 - 1) + col);
    Vc = load_prim_at(plane_of(m0) + col);
    Vp1 = load_prim_at(plane_of(m0 + 1) + col);
    load_fields<Real, NF>(Uin, N, plane_of(m0 + 2) + col, Unext);
    P him1, loc;
    interpolate<Real, D>(Vm2, Vm1, Vc, nullptr, &him1);
    interpolate<Real, D>(Vm1, Vc, Vp1, &loc, &hiM);
    riemann_flux<Real, D, M, RS>(g.gamma, g.igm1, him1, loc, Fprev);
    sts_plane(0, lj + OY, li + 2, Vc);
    if (is_halo) {
      sts_plane(0, hpy + OY, hpx + 2, load_prim_at(plane_of(m0) + hcol));
      if (m0 + 1 < m1) load_fields<Real, NF>(Uin, N, plane_of(m0 + 1) + hcol, Uh);
    }
  }
  __syncthreads();

  Real s_max = Real(0);
  int bad = 0;
  int b = 0;
  for (int m = m0; m < m1; ++m, b ^= 1) {
    // ------------------------------------------------------------ phase A
    // own-cell base state of Eq. 23 (coherent load: the last stage overwrites U_base in place)
    Real u[NF];
    if (active) load_fields_rw<Real, NF>(Ubase, N, plane_of(m) + own, u);

    // in-plane reconstruction of the own cell (Eq. 20-21), lo handed to the lower neighbour
    P hix, hiy;
    {
      P lo;
      interpolate<Real, D>(lds_plane(b, lj + OY, li + 1), Vc, lds_plane(b, lj + OY, li + 3), &lo, &hix);
      Real a[NF];
      prim_to_array<Real, D>(lo, a);
#pragma unroll
      for (int f = 0; f < NF; ++f) sm.Ex[f][lj][li] = a[f];
      if constexpr (D == 3) {
        interpolate<Real, D>(lds_plane(b, lj + 1, li + 2), Vc, lds_plane(b, lj + 3, li + 2), &lo, &hiy);
        prim_to_array<Real, D>(lo, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) sm.Ey[f][lj][li] = a[f];
      }
    }
    // halo tasks, part 1: lo of the first cell beyond the tile
    if (t >= XTASK0 && t < XTASK0 + TY) {
      const int r = t - XTASK0;
      P lo;
      interpolate<Real, D>(lds_plane(b, r + OY, TX + 1), lds_plane(b, r + OY, TX + 2), lds_plane(b, r + OY, TX + 3), &lo,
                           nullptr);
      Real a[NF];
      prim_to_array<Real, D>(lo, a);
#pragma unroll
      for (int f = 0; f < NF; ++f) sm.Ex[f][r][TX] = a[f];
    }
    if constexpr (D == 3) {
      if (t >= YTASK0) {
        const int c = t - YTASK0;
        P lo;
        interpolate<Real, D>(lds_plane(b, TY + 1, c + 2), lds_plane(b, TY + 2, c + 2), lds_plane(b, TY + 3, c + 2), &lo,
                             nullptr);
        Real a[NF];
        prim_to_array<Real, D>(lo, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) sm.Ey[f][TY][c] = a[f];
      }
    }

    // marching axis: V[m+2], slope of cell m+1, flux through face m+1/2
    const P Vp2 = prim_of<Real, D>(Unext, g.gm1);
    if (m + 1 < m1) load_fields<Real, NF>(Uin, N, plane_of(m + 3) + col, Unext);
    P loM1, hiM1;
    interpolate<Real, D>(Vc, Vp1, Vp2, &loM1, &hiM1);
    Real Fnext[NF];
    riemann_flux<Real, D, M, RS>(g.gamma, g.igm1, hiM, loM1, Fnext);

    // primitives of the next plane into the other buffer
    if (m + 1 < m1) {
      sts_plane(b ^ 1, lj + OY, li + 2, Vp1);
      if (is_halo) {
        sts_plane(b ^ 1, hpy + OY, hpx + 2, prim_of<Real, D>(Uh, g.gm1));
        if (m + 2 < m1) load_fields<Real, NF>(Uin, N, plane_of(m + 2) + hcol, Uh);
      }
    }
    __syncthreads();

    // ------------------------------------------------------------ phase B: one Riemann solve per face
    Real Fx[NF], Fy[NF];
    {
      Real a[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) a[f] = sm.Ex[f][lj][li + 1];
      riemann_flux<Real, D, 0, RS>(g.gamma, g.igm1, hix, prim_from_array<Real, D>(a), Fx);
#pragma unroll
      for (int f = 0; f < NF; ++f) sm.Ex[f][lj][li + 1] = Fx[f];
      if constexpr (D == 3) {
#pragma unroll
        for (int f = 0; f < NF; ++f) a[f] = sm.Ey[f][lj + 1][li];
        riemann_flux<Real, D, 1, RS>(g.gamma, g.igm1, hiy, prim_from_array<Real, D>(a), Fy);
#pragma unroll
        for (int f = 0; f < NF; ++f) sm.Ey[f][lj + 1][li] = Fy[f];
      }
    }
    // halo tasks, part 2: flux through the tile's lowest face
    if (t >= XTASK0 && t < XTASK0 + TY) {
      const int r = t - XTASK0;
      P hi;
      interpolate<Real, D>(lds_plane(b, r + OY, 0), lds_plane(b, r + OY, 1), lds_plane(b, r + OY, 2), nullptr, &hi);
      Real a[NF], F[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) a[f] = sm.Ex[f][r][0];
      riemann_flux<Real, D, 0, RS>(g.gamma, g.igm1, hi, prim_from_array<Real, D>(a), F);
#pragma unroll
      for (int f = 0; f < NF; ++f) sm.Ex[f][r][0] = F[f];
    }
    if constexpr (D == 3) {
      if (t >= YTASK0) {
        const int c = t - YTASK0;
        P hi;
        interpolate<Real, D>(lds_plane(b, 0, c + 2), lds_plane(b, 1, c + 2), lds_plane(b, 2, c + 2), nullptr, &hi);
        Real a[NF], F[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) a[f] = sm.Ey[f][0][c];
        riemann_flux<Real, D, 1, RS>(g.gamma, g.igm1, hi, prim_from_array<Real, D>(a), F);
#pragma unroll
        for (int f = 0; f < NF; ++f) sm.Ey[f][0][c] = F[f];
      }
    }
    __syncthreads();

    // ------------------------------------------------------------ phase C: Eq. 23, axes in the order x, y, z
    if (active) {
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = rfma(lam0, sm.Ex[f][lj][li] - Fx[f], u[f]);
      if constexpr (D == 3) {
#pragma unroll
        for (int f = 0; f < NF; ++f) u[f] = rfma(lam1, sm.Ey[f][lj][li] - Fy[f], u[f]);
#pragma unroll
        for (int f = 0; f < NF; ++f) u[f] = rfma(lam2, Fprev[f] - Fnext[f], u[f]);
      } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) u[f] = rfma(lam1, Fprev[f] - Fnext[f], u[f]);
      }
      if (STAGE == 2 && g.integrator == 1) {  // Heun: U2 = 0.5 (U0 + (U1 + dt L(U1))); U0 still sits in Uout
        Real u0[NF];
        load_fields_rw<Real, NF>(Uout, N, plane_of(m) + own, u0);
#pragma unroll
        for (int f = 0; f < NF; ++f) u[f] = Real(0.5) * (u0[f] + u[f]);
      }
      store_fields<Real, NF>(Uout, N, plane_of(m) + own, u);
      if (STAGE == 2) {
        Real ir;
        const P Vn = prim_of<Real, D>(u, g.gm1, &ir);
        s_max = rmax(s_max, cfl_speed<Real, D>(Vn, ir, g.gamma, g.idr));
        bad += bad_state<Real, D>(Vn, u[NF - 1]);
      }
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) Fprev[f] = Fnext[f];
    Vc = Vp1;
    Vp1 = Vp2;
    hiM = hiM1;
  }
  if (STAGE == 2) {
    const unsigned int nblocks = gridDim.x * gridDim.y * gridDim.z;
    block_reduce_and_finalize<Real>(s_max, bad, sc, g, nblocks, 1);
  }
}

// ------------------------------------------------------------------------------------------------
template <class Real, int D, int RS, int STAGE, int TX, int TY>
static bool launch_fused_shape(const Real* Uin, const Real* Ubase, Real* Uout, const Geom<Real>& g, Scalars* sc,
                               cudaStream_t stream, int depth) {
  using Smem = FusedSmem<Real, D, TX, TY>;
  auto kern = k_fused<Real, D, RS, STAGE, TX, TY>;
  // the opt-in to more than 48 KB of dynamic shared memory is a per-device attribute of the kernel
  static bool configured[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
  if (!configured[dev]) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)) != cudaSuccess)
      return false;
    configured[dev] = true;
  }
  constexpr int M = D - 1;
  dim3 grid, block(TX, TY, 1);
  grid.x = (g.n[0] + TX - 1) / TX;
  if (D == 3) {
    grid.y = (g.n[1] + TY - 1) / TY;
    grid.z = (g.n[M] + depth - 1) / depth;
    if (grid.y > 65535u || grid.z > 65535u) return false;
  } else {
    grid.y = (g.n[M] + depth - 1) / depth;
    grid.z = 1;
    if (grid.y > 65535u) return false;
  }
  kern<<<grid, block, sizeof(Smem), stream>>>(Uin, Ubase, Uout, g, sc, depth);
  return true;
}

// Tile depth when the caller gives none: deep enough that the 4 extra planes of primitives and the extra
// face per tile stay below ~10 % of the work, shallow enough to give every SM several blocks.
inline int default_tile_depth(long long tiles_in_plane, int nM) {
  int depth = 32;
  while (depth > 8 && tiles_in_plane * ((nM + depth - 1) / depth) < 4 * device_sm_count()) depth >>= 1;
  return depth;
}

// Returns false when the marching kernel does not cover this shape (the caller then uses k_delayed).
//   block[0], block[1]: tile shape TX x TY (0 = default); tile_depth: planes marched per block (0 = default)
template <class Real, int D, int RS, int STAGE>
bool launch_fused_stage(const Real* Uin, const Real* Ubase, Real* Uout, const Geom<Real>& g, Scalars* sc,
                        cudaStream_t stream, const int* block, int tile_depth) {
  if constexpr (D == 1) {
    return false;
  } else if constexpr (D == 2) {
    int tx = block[0] > 0 ? block[0] : 128;  // 256-thread rows of the fp64 last stage need 148 registers: one block per SM
    const long long tiles = (g.n[0] + tx - 1) / tx;
    const int depth = tile_depth > 0 ? tile_depth : default_tile_depth(tiles, g.n[1]);
#define PH_SHAPE(TXV) \
  if (tx == TXV) return launch_fused_shape<Real, D, RS, STAGE, TXV, 1>(Uin, Ubase, Uout, g, sc, stream, depth);
    PH_SHAPE(64) PH_SHAPE(128) PH_SHAPE(256) PH_SHAPE(512)
#undef PH_SHAPE
    return false;
  } else {
    const int tx = block[0] > 0 ? block[0] : 32;
    const int ty = block[1] > 0 ? block[1] : 8;
    const long long tiles = (long long)((g.n[0] + tx - 1) / tx) * ((g.n[1] + ty - 1) / ty);
    const int depth = tile_depth > 0 ? tile_depth : default_tile_depth(tiles, g.n[2]);
#define PH_SHAPE(TXV, TYV) \
  if (tx == TXV && ty == TYV) \
    return launch_fused_shape<Real, D, RS, STAGE, TXV, TYV>(Uin, Ubase, Uout, g, sc, stream, depth);
    PH_SHAPE(32, 8) PH_SHAPE(32, 16) PH_SHAPE(64, 8)
#undef PH_SHAPE
    return false;
  }
}

}  // namespace ph
