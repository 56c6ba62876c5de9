// hydro_kernels_march.cuh — the fused RK-stage kernel, second design ("march"): ONE kernel per RK stage,
// every intermediate on chip and computed once per cell / face (Fig. 6-7 :435-472 rebuilt for
// sm_100a), organised around what the r1b Nsight capture of k_fused showed (profiles/r1b_README.md):
// the stage is bound by instruction issue, not by DRAM.
//
//   * T = float / double: one cell per thread and x position (the default).  T = f32x2 (option cells_per_thread
//     = 2): a thread owns TWO x-adjacent cells, held in 64-bit register pairs and computed with the packed
//     FADD2 / FMUL2 / FFMA2 instructions (one issue slot, two IEEE-rounded fp32 results, bit-identical to the
//     scalar instructions), 64-bit global and shared accesses; fewer instructions per cell but ~210 registers:
//     measured slower, kept as an option.  Further options of the same kind: RPT = 2 (two
//     y-adjacent cells per thread), TMA (bulk-copy staging of the tile rows into a shared-memory ring).
//   * a block = NWX x TY "main" warps (a tile of TXC = NWX*32*W cells by TY rows of the leading plane, marched
//     through `depth` planes of the last axis with a rolling register window, as in k_fused) + ONE halo warp.
//     The halo warp loads the 2-cell star halo of every plane, converts it to primitives, and computes the
//     faces the tile cannot get from its own cells (the flux through the tile's low x / y faces, the low-side
//     state of the first cell beyond its high x / y faces), so the main warps all do the same work and the two
//     block barriers per plane no longer wait for stragglers.
//   * x-neighbours inside a warp exchange face states and fluxes by warp shuffle; only warp-edge lanes and the
//     y direction go through shared memory.
//   * Eq. 23 is applied in the order x, y, z onto U_base (R11); the last stage forms the primitives
//     of the new state in registers and feeds the CFL max (a0) into the block reduction.
// Ragged tiles and periodic / outflow ghosts need no special cases: a plane position whose global index g lies
// outside [0, n) holds the state of a mapped cell (wrap or clamp); threads whose own cells lie outside the grid
// compute but never store.  T = f32x2 needs an even n_x (the launcher falls back to T = float otherwise).
#pragma once
#include <cuda.h>  // CUtensorMap (the descriptor of the tensor-map TMA staging, TMA = 2)

#include <cstring>

#include "hydro_kernels_basic.cuh"

// blocks per SM the register cap of __launch_bounds__ is set for: fp32 one cell per thread (two 256-thread blocks,
// <= 128 registers), and the two-rows-per-thread shape (one block)
#ifndef PH_RPT2_MINB
#define PH_RPT2_MINB 1
#endif
#ifndef PH_MARCH_MINB
#define PH_MARCH_MINB 2
#endif

namespace ph {

// ---------------------------------------------------------------- lane helpers
__device__ __forceinline__ float lane_first(float a) { return a; }
__device__ __forceinline__ double lane_first(double a) { return a; }
__device__ __forceinline__ float lane_first(f32x2 a) { return a.v.x; }
__device__ __forceinline__ float lane_first(f32fast a) { return a.v; }
__device__ __forceinline__ float lane_last(f32fast a) { return a.v; }
__device__ __forceinline__ f32fast xshift_left(f32fast, float nb) { return f32fast(nb); }
__device__ __forceinline__ f32fast xshift_right(f32fast, float nb) { return f32fast(nb); }
__device__ __forceinline__ f32fast lane_pack(float a, float, f32fast*) { return f32fast(a); }
__device__ __forceinline__ float lane_last(float a) { return a; }
__device__ __forceinline__ double lane_last(double a) { return a; }
__device__ __forceinline__ float lane_last(f32x2 a) { return a.v.y; }
__device__ __forceinline__ void lane_set_last(float& a, float x) { a = x; }
__device__ __forceinline__ void lane_set_last(double& a, double x) { a = x; }
__device__ __forceinline__ void lane_set_last(f32x2& a, float x) { a.v.y = x; }
// the x-neighbour views of a thread's cells: (left neighbour, own cells but the last) / (own cells but the first, right)
__device__ __forceinline__ float xshift_left(float, float nb) { return nb; }
__device__ __forceinline__ double xshift_left(double, double nb) { return nb; }
__device__ __forceinline__ f32x2 xshift_left(f32x2 own, float nb) { return f32x2(nb, own.v.x); }
__device__ __forceinline__ float xshift_right(float, float nb) { return nb; }
__device__ __forceinline__ double xshift_right(double, double nb) { return nb; }
__device__ __forceinline__ f32x2 xshift_right(f32x2 own, float nb) { return f32x2(own.v.y, nb); }
// two independent scalars as the lanes of one value (W = 1: the first only)
__device__ __forceinline__ float lane_pack(float a, float, float*) { return a; }
__device__ __forceinline__ double lane_pack(double a, double, double*) { return a; }
__device__ __forceinline__ f32x2 lane_pack(float a, float b, f32x2*) { return f32x2(a, b); }

template <class T> __device__ __forceinline__ T lds(const scalar_t<T>* p) { return *p; }
template <> __device__ __forceinline__ f32x2 lds<f32x2>(const float* p) { return f32x2(*reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ void sts(float* p, float v) { *p = v; }
__device__ __forceinline__ void sts(float* p, f32fast v) { *p = v.v; }
__device__ __forceinline__ void sts(double* p, double v) { *p = v; }
__device__ __forceinline__ void sts(float* p, f32x2 v) { *reinterpret_cast<float2*>(p) = v.v; }

template <class T, int D>
__device__ __forceinline__ Prim<T, D> prim_from_fields(const T (&u)[D + 2]) {
  Prim<T, D> P;
  P.rho = u[0];
#pragma unroll
  for (int b = 0; b < D; ++b) P.v[b] = u[1 + b];
  P.p = u[D + 1];
  return P;
}
template <class T, int D>
__device__ __forceinline__ void prim_to_fields(const Prim<T, D>& P, T (&u)[D + 2]) {
  u[0] = P.rho;
#pragma unroll
  for (int b = 0; b < D; ++b) u[1 + b] = P.v[b];
  u[D + 1] = P.p;
}

// flags lanes whose new state is unusable (R19)
template <class T, int D>
__device__ __forceinline__ int bad_lanes(const Prim<T, D>& V, T E) {
  using S = scalar_t<T>;
  const T zero = T(S(0));
  return lane_count(m_or(m_or(m_not(gt(V.rho, zero)), m_not(gt(V.p, zero))), m_not(le(rabs(E), T(S(3.0e38))))));
}

// TMA: 0 none | 1 bulk row copies (cp.async.bulk, SASS UBLKCP) | 2 one tensor-map copy per plane (cp.async.bulk.tensor, UTMALDG)
template <class T, int D, int NWX, int TY, int TMA = 0, int RPT = 1>
struct MarchShape {
  using S = scalar_t<T>;
  static constexpr int W = LaneTraits<T>::W;
  static constexpr int NF = D + 2;
  static constexpr int TXC = NWX * 32 * W;              // cells per tile row
  static constexpr int PX = TXC + 4;                    // plane row: tile + 2 halo cells on each side
  static constexpr int TYC = TY * RPT;                  // tile rows: RPT rows per main warp
  static constexpr int PY = (D == 3) ? TYC + 4 : 1;
  static constexpr int OY = (D == 3) ? 2 : 0;           // plane row of the tile's first row
  static constexpr int NMAIN = NWX * TY * 32;           // main threads; the halo warp follows them
  static constexpr int NT = NMAIN + 32;
  static constexpr int XROWS = (D == 3) ? TYC : 1;      // tile rows = x halo tasks per plane
  static constexpr int XTASK_LANES = (XROWS + W - 1) / W;
  static constexpr int XHALO_LANES = 4 * XROWS / W;     // lanes of the halo warp that load x halo cells
  static_assert(D == 2 || D == 3, "the marching kernel covers 2-D and 3-D grids");
  static_assert(D == 3 || TY == 1, "2-D tiles are rows");
  static_assert(D == 2 || NWX == 1, "3-D tiles are one warp wide");
  static_assert(RPT == 1 || (D == 3 && RPT == 2 && !TMA), "two rows per thread: 3-D, per-thread loads");
  static_assert(XTASK_LANES <= 32, "tile too tall for one halo warp");
  static constexpr int RING = 4;                        // TMA: raw planes m .. m+3 of the tile's own cells
  struct Smem {
    // TMA staging (bulk async copies, one per tile row and field, complete on an mbarrier): the conserved state of
    // the tile's own cells, planes m .. m+3 of U_in (stage 1 takes U_base from the same ring) and, for the last
    // stage, planes m, m+1 of U_base = U0.  Rows are 16-byte aligned: first members of a 128-byte aligned struct.
    S Uraw[TMA ? RING : 1][TMA ? NF : 1][TMA ? XROWS : 1][TMA ? TXC : 4];
    S Ub[TMA ? 2 : 1][TMA ? NF : 1][TMA ? XROWS : 1][TMA ? TXC : 4];
    unsigned long long mbar[RING + 2];
    S V[2][NF][PY][PX];                                 // primitives of plane m (double-buffered), halo 2
    S LOy[(D == 3) ? NF : 1][TYC + 1][(D == 3) ? TXC : 2];  // [r]: low-side y state of tile row r (r = TYC: halo warp)
    S Fy[(D == 3) ? NF : 1][TYC][(D == 3) ? TXC : 2];   // [r]: flux through the low y face of tile row r (r = 0: halo warp)
    S LOx[NF][XROWS][NWX + 1];                          // [e]: low-side x state of the first cell of warp column e (e = NWX: halo warp)
    S Fx[NF][XROWS][NWX];                               // [e]: flux through the low x face of warp column e (e = 0: halo warp)
  };
};

// position g of a plane axis -> the cell whose state it holds (g >= -2)
__device__ __forceinline__ int march_src(int g, int n, int boundary) {
  return map_index(g > n + 1 ? n + 1 : g, n, boundary);
}

// Where the W cells at x positions g .. g+W-1 (g even for W = 2) of a grid row come from: element offsets inside
// a plane, fixed for the whole march (only the plane changes), so that the index mapping is done once per thread.
struct CellSrc {
  int o0, o1;   // first / second cell (o1 unused for W = 1)
  bool pair;    // W = 2: the two cells are adjacent in memory and 8-byte aligned -> one 64-bit load
};
template <class T>
__device__ __forceinline__ CellSrc cell_src(int g, int rowoff, int nx, int bnd) {
  CellSrc c;
  if constexpr (LaneTraits<T>::W == 1) {
    c.o0 = c.o1 = rowoff + march_src(g, nx, bnd);
    c.pair = false;
  } else if (bnd == BOUNDARY_PERIODIC) {
    int gp = g > nx ? nx : g;  // nx even: (gp, gp+1) wraps as a pair
    gp = gp < 0 ? gp + nx : (gp >= nx ? gp - nx : gp);
    c.o0 = rowoff + gp;
    c.o1 = c.o0 + 1;
    c.pair = true;
  } else {
    c.o0 = rowoff + march_src(g, nx, bnd);
    c.o1 = rowoff + march_src(g + 1, nx, bnd);
    c.pair = g >= 0 && g + 1 < nx;
  }
  return c;
}
// base = element index of the first cell of one field of one plane (all indices fit an int: nf*N < 2^31)
template <class T>
__device__ __forceinline__ T ldg_cells(const scalar_t<T>* __restrict__ A, int base, const CellSrc& c) {
  if constexpr (LaneTraits<T>::W == 1) {
    return __ldg(A + (base + c.o0));
  } else {
    if (c.pair) return f32x2(__ldg(reinterpret_cast<const float2*>(A + (base + c.o0))));
    return f32x2(__ldg(A + (base + c.o0)), __ldg(A + (base + c.o1)));
  }
}
template <class T>
__device__ __forceinline__ T ld_cells_rw(const scalar_t<T>* A, int idx) {
  if constexpr (LaneTraits<T>::W == 1) return A[idx];
  else return f32x2(*reinterpret_cast<const float2*>(A + idx));
}
__device__ __forceinline__ float scalar_of(float v) { return v; }
__device__ __forceinline__ double scalar_of(double v) { return v; }
__device__ __forceinline__ float scalar_of(f32fast v) { return v.v; }
template <class T>
__device__ __forceinline__ void st_cells(scalar_t<T>* A, int idx, T v) {
  if constexpr (LaneTraits<T>::W == 1) A[idx] = scalar_of(v);
  else *reinterpret_cast<float2*>(A + idx) = v.v;
}
__device__ __forceinline__ float shfl_dn(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_up(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_up(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// All warps of the block arrive at barrier 0 the same number of times, the main warps and the halo warp from
// different places in the code (PTX bar.sync semantics: arrival is counted per warp, not per call site).
// ---------------------------------------------------------------- TMA bulk copies completing on an mbarrier
__device__ __forceinline__ unsigned int smem_addr(const void* p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, int bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned int parity) {
  unsigned int done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_addr(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned (cp.async.bulk: SASS UBLKCP)
__device__ __forceinline__ void tma_row(void* dst, const void* src, int bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr(dst)),
               "l"(src), "r"(bytes), "r"(smem_addr(bar))
               : "memory");
}

__device__ __forceinline__ void block_barrier() { asm volatile("bar.sync 0;" ::: "memory"); }

// global -> shared, one box of a tensor map (cp.async.bulk.tensor: SASS UTMALDG); rank 3 (x, y, f) or 4 (x, y, z, f)
__device__ __forceinline__ void tma_box3(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                   smem_addr(dst)),
               "l"(reinterpret_cast<unsigned long long>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_addr(bar))
               : "memory");
}
__device__ __forceinline__ void tma_box4(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
                   smem_addr(dst)),
               "l"(reinterpret_cast<unsigned long long>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_addr(bar))
               : "memory");
}

template <class T, int D, int RS, int STAGE, int NWX, int TY, int MINB, int TMA, int RPT>
__global__ void __launch_bounds__(MarchShape<T, D, NWX, TY, TMA, RPT>::NT, MINB)
    k_march(const scalar_t<T>* __restrict__ Uin, const scalar_t<T>* Ubase, scalar_t<T>* Uout, Geom<scalar_t<T>> g,
            Scalars* sc, int depth, const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_base) {
  using Sh = MarchShape<T, D, NWX, TY, TMA, RPT>;
  using S = scalar_t<T>;
  using P = Prim<T, D>;
  constexpr int W = Sh::W, NF = Sh::NF, TXC = Sh::TXC, OY = Sh::OY, XROWS = Sh::XROWS, TYC = Sh::TYC;
  constexpr int M = D - 1;  // marching axis
  constexpr int RING = Sh::RING;

  if (sc->done) return;
  extern __shared__ __align__(128) unsigned char march_smem_raw[];
  typename Sh::Smem& sm = *reinterpret_cast<typename Sh::Smem*>(march_smem_raw);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nx = g.n[0], ny = g.n[1], nM = g.n[M], bnd = g.boundary;
  const int x0 = blockIdx.x * TXC;
  const int y0 = (D == 3) ? blockIdx.y * TYC : 0;
  const int bm = (D == 3) ? blockIdx.z : blockIdx.y;
  const int m0 = bm * depth;
  const int m1 = min(m0 + depth, nM);
  const int Ni = int(g.N);                              // every element index fits an int: nf*N < 2^31 (create)
  const int psi = (D == 3) ? nx * ny : nx;              // cells per plane
  auto plane_of = [&](int m) { return map_index(m, nM, bnd) * psi; };
  auto grid_row = [&](int gj) { return (D == 3) ? march_src(gj, ny, bnd) * nx : 0; };

  // TMA staging needs whole, 16-byte aligned rows: tiles that end inside the grid (the launcher checks n_x % 4)
  // (TMA = 2: a box does not wrap, so the tile's rows must lie inside the grid as well)
  const bool use_tma = TMA && (x0 + TXC <= nx) && (TMA == 1 || D == 2 || y0 + TYC <= ny);

  S s_max = S(0);
  int bad = 0;

  if (warp < NWX * TY) {
    // =========================================================================== main warps
    // A thread owns RPT cells of one x position: tile rows RPT*warp .. RPT*warp + RPT-1 (3-D; RPT = 1 in 2-D).  With
    // RPT = 2 the y face between its two cells never leaves the registers and the halo warp serves twice the rows.
    const int wx = (D == 3) ? 0 : warp;
    const int c0 = (wx * 32 + lane) * W;  // first own cell, tile coordinates
    const int gi = x0 + c0;
    const int pc = c0 + 2;                // own column in the shared plane
    int row[RPT], pr[RPT], own[RPT];
    bool active[RPT];
    CellSrc src[RPT];
#pragma unroll
    for (int rr = 0; rr < RPT; ++rr) {
      row[rr] = (D == 3) ? warp * RPT + rr : 0;
      const int gj = y0 + row[rr];
      active[rr] = gi < nx && (D == 2 || gj < ny);
      src[rr] = cell_src<T>(gi, grid_row(gj), nx, bnd);
      own[rr] = (D == 3 ? gj * nx : 0) + gi;  // valid when active
      pr[rr] = row[rr] + OY;
    }

    auto load_cells_of = [&](const CellSrc& c, int m, T (&u)[NF]) {
      const int pl = plane_of(m);
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = ldg_cells<T>(Uin, f * Ni + pl, c);
    };
    auto sts_plane = [&](int b, int py, const P& V) {
      T u[NF];
      prim_to_fields<T, D>(V, u);
#pragma unroll
      for (int f = 0; f < NF; ++f) sts(&sm.V[b][f][py][pc], u[f]);
    };
    auto lds_plane = [&](int b, int py) {
      T u[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = lds<T>(&sm.V[b][f][py][pc]);
      return prim_from_fields<T, D>(u);
    };

    const S lam0 = S(sc->lam[STAGE - 1][0]);
    const S lam1 = S(sc->lam[STAGE - 1][1]);
    const S lam2 = (D == 3) ? S(sc->lam[STAGE - 1][2]) : S(0);

    // ---- prologue: rolling window at m0
    P Vc[RPT], Vp1[RPT], hiM[RPT];
    T Fprev[RPT][NF], Unext[RPT][NF];
#pragma unroll
    for (int rr = 0; rr < RPT; ++rr) {
      T u[NF];
      load_cells_of(src[rr], m0 - 2, u);
      const P Vm2 = prim_of<T, D>(u, g.gm1);
      load_cells_of(src[rr], m0 - 1, u);
      const P Vm1 = prim_of<T, D>(u, g.gm1);
      load_cells_of(src[rr], m0, u);
      Vc[rr] = prim_of<T, D>(u, g.gm1);
      load_cells_of(src[rr], m0 + 1, u);
      Vp1[rr] = prim_of<T, D>(u, g.gm1);
      if (!use_tma) load_cells_of(src[rr], m0 + 2, Unext[rr]);
      P him1, loc;
      interpolate<T, D>(Vm2, Vm1, Vc[rr], nullptr, &him1);
      interpolate<T, D>(Vm1, Vc[rr], Vp1[rr], &loc, &hiM[rr]);
      riemann_flux<T, D, M, RS>(g.gamma, g.igm1, him1, loc, Fprev[rr]);
      sts_plane(0, pr[rr], Vc[rr]);
    }
    block_barrier();

    int b = 0;
    for (int m = m0; m < m1; ++m, b ^= 1) {
      const bool more = m + 1 < m1;
      const int q = m - m0;  // plane index inside this block's march
      // ------------------------------------------------------------ phase A: slopes, the marching-axis face
      P hix[RPT], lox[RPT], hiy[RPT], loy_up;  // loy_up (RPT = 2): low-side y state of the thread's upper cell
#pragma unroll
      for (int rr = 0; rr < RPT; ++rr) {
        T vc[NF], l[NF], r[NF];
        prim_to_fields<T, D>(Vc[rr], vc);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          l[f] = xshift_left(vc[f], sm.V[b][f][pr[rr]][pc - 1]);
          r[f] = xshift_right(vc[f], sm.V[b][f][pr[rr]][pc + W]);
        }
        interpolate<T, D>(prim_from_fields<T, D>(l), Vc[rr], prim_from_fields<T, D>(r), &lox[rr], &hix[rr]);
        if (lane == 0) {  // low-side state of this warp column's first cell, for the warp (or halo task) on its left
          T a[NF];
          prim_to_fields<T, D>(lox[rr], a);
#pragma unroll
          for (int f = 0; f < NF; ++f) sm.LOx[f][row[rr]][wx] = lane_first(a[f]);
        }
      }
      if constexpr (D == 3) {
        // y slopes: neighbours inside the thread come from registers, the others from the shared plane
        P loy;
        if constexpr (RPT == 1) {
          interpolate<T, D>(lds_plane(b, pr[0] - 1), Vc[0], lds_plane(b, pr[0] + 1), &loy, &hiy[0]);
        } else {
          interpolate<T, D>(lds_plane(b, pr[0] - 1), Vc[0], Vc[1], &loy, &hiy[0]);
          interpolate<T, D>(Vc[0], Vc[1], lds_plane(b, pr[1] + 1), &loy_up, &hiy[1]);
        }
        T a[NF];
        prim_to_fields<T, D>(loy, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) sts(&sm.LOy[f][row[0]][c0], a[f]);
      }
      // marching axis: V[m+2], slope of cell m+1, flux through face m+1/2
      P Vp2[RPT], hiM1[RPT];
      T Fnext[RPT][NF];
#pragma unroll
      for (int rr = 0; rr < RPT; ++rr) {
        if (TMA && use_tma) {  // U_in of plane m+2: landed in ring slot (q+2) % RING one iteration ago
          mbar_wait(&sm.mbar[(q + 2) % RING], ((q + 2) / RING) & 1);
#pragma unroll
          for (int f = 0; f < NF; ++f) Unext[rr][f] = lds<T>(&sm.Uraw[(q + 2) % RING][f][row[rr]][c0]);
        }
        Vp2[rr] = prim_of<T, D>(Unext[rr], g.gm1);
        if (more && !use_tma) load_cells_of(src[rr], m + 3, Unext[rr]);
        P loM1;
        interpolate<T, D>(Vc[rr], Vp1[rr], Vp2[rr], &loM1, &hiM1[rr]);
        riemann_flux<T, D, M, RS>(g.gamma, g.igm1, hiM[rr], loM1, Fnext[rr]);
        if (more) sts_plane(b ^ 1, pr[rr], Vp1[rr]);
      }
      block_barrier();

      // ------------------------------------------------------------ phase B: one Riemann solve per in-plane face
      T Fx[RPT][NF], Fy[RPT][NF];  // Fy[rr]: flux through the upper y face of the thread's cell rr
#pragma unroll
      for (int rr = 0; rr < RPT; ++rr) {
        T a[NF], rs[NF];
        prim_to_fields<T, D>(lox[rr], a);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          S nb = shfl_dn(lane_first(a[f]));
          if (lane == 31) nb = sm.LOx[f][row[rr]][wx + 1];
          rs[f] = xshift_right(a[f], nb);
        }
        riemann_flux<T, D, 0, RS>(g.gamma, g.igm1, hix[rr], prim_from_fields<T, D>(rs), Fx[rr]);
        if (NWX > 1 && lane == 31 && wx + 1 < NWX) {
#pragma unroll
          for (int f = 0; f < NF; ++f) sm.Fx[f][row[rr]][wx + 1] = lane_last(Fx[rr][f]);
        }
      }
      if constexpr (D == 3) {
        if constexpr (RPT == 2) riemann_flux<T, D, 1, RS>(g.gamma, g.igm1, hiy[0], loy_up, Fy[0]);
        T a[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) a[f] = lds<T>(&sm.LOy[f][row[RPT - 1] + 1][c0]);
        riemann_flux<T, D, 1, RS>(g.gamma, g.igm1, hiy[RPT - 1], prim_from_fields<T, D>(a), Fy[RPT - 1]);
        if (row[RPT - 1] + 1 < TYC) {
#pragma unroll
          for (int f = 0; f < NF; ++f) sts(&sm.Fy[f][row[RPT - 1] + 1][c0], Fy[RPT - 1][f]);
        }
      }
      // own-cell base state of Eq. 23 (coherent load: the last stage overwrites U_base in place)
      const int pl = plane_of(m);
      T u[RPT][NF];
#pragma unroll
      for (int rr = 0; rr < RPT; ++rr) {
        if (TMA && use_tma) {  // stage 1: U_base = U_in, plane m of the ring; last stage: the U0 ring
          if (STAGE == 1) {
            mbar_wait(&sm.mbar[q % RING], (q / RING) & 1);
#pragma unroll
            for (int f = 0; f < NF; ++f) u[rr][f] = lds<T>(&sm.Uraw[q % RING][f][row[rr]][c0]);
          } else {
            mbar_wait(&sm.mbar[RING + (q & 1)], (q >> 1) & 1);
#pragma unroll
            for (int f = 0; f < NF; ++f) u[rr][f] = lds<T>(&sm.Ub[q & 1][f][row[rr]][c0]);
          }
        } else if (active[rr]) {
#pragma unroll
          for (int f = 0; f < NF; ++f) u[rr][f] = ld_cells_rw<T>(Ubase, f * Ni + pl + own[rr]);
        }
      }
      block_barrier();

      // ------------------------------------------------------------ phase C: Eq. 23, axes in the order x, y, z
#pragma unroll
      for (int rr = 0; rr < RPT; ++rr) {
        T lowx[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          S nb = shfl_up(lane_last(Fx[rr][f]));
          if (lane == 0) nb = sm.Fx[f][row[rr]][wx];
          lowx[f] = xshift_left(Fx[rr][f], nb);
        }
        if (active[rr]) {
          const int cell = pl + own[rr];
#pragma unroll
          for (int f = 0; f < NF; ++f) u[rr][f] = rfma(lam0, lowx[f] - Fx[rr][f], u[rr][f]);
          if constexpr (D == 3) {
#pragma unroll
            for (int f = 0; f < NF; ++f) {
              const T lowy = (rr == 0) ? lds<T>(&sm.Fy[f][row[0]][c0]) : Fy[0][f];
              u[rr][f] = rfma(lam1, lowy - Fy[rr][f], u[rr][f]);
            }
#pragma unroll
            for (int f = 0; f < NF; ++f) u[rr][f] = rfma(lam2, Fprev[rr][f] - Fnext[rr][f], u[rr][f]);
          } else {
#pragma unroll
            for (int f = 0; f < NF; ++f) u[rr][f] = rfma(lam1, Fprev[rr][f] - Fnext[rr][f], u[rr][f]);
          }
          if (STAGE == 2 && g.integrator == 1) {  // Heun: U2 = 0.5 (U0 + (U1 + dt L(U1))); U0 still sits in Uout
#pragma unroll
            for (int f = 0; f < NF; ++f) u[rr][f] = S(0.5) * (ld_cells_rw<T>(Uout, f * Ni + cell) + u[rr][f]);
          }
#pragma unroll
          for (int f = 0; f < NF; ++f) st_cells<T>(Uout, f * Ni + cell, u[rr][f]);
          if (STAGE == 2) {
            T ir;
            const P Vn = prim_of<T, D>(u[rr], g.gm1, &ir);
            s_max = rmax(s_max, lane_max(cfl_speed<T, D>(Vn, ir, g.gamma, g.idr)));
            bad += bad_lanes<T, D>(Vn, u[rr][NF - 1]);
          }
        }
#pragma unroll
        for (int f = 0; f < NF; ++f) Fprev[rr][f] = Fnext[rr][f];
        Vc[rr] = Vp1[rr];
        Vp1[rr] = Vp2[rr];
        hiM[rr] = hiM1[rr];
      }
    }
  } else {
    // =========================================================================== the halo warp
    // It loads the whole 2-cell star halo of every plane (x halo cells and y halo rows), converts it to primitives and
    // computes the faces the tile cannot get from its own cells.  Its face tasks read only the shared plane and
    // the low-side states the main warps publish, so it never waits for anything but the block barriers.
    constexpr int NXP = (Sh::XHALO_LANES + 31) / 32;  // x halo slots per lane
    CellSrc hsrc[NXP];
    int hpy[NXP], hpx[NXP];
    bool hval[NXP];
#pragma unroll
    for (int q = 0; q < NXP; ++q) {
      const int id = lane + 32 * q;
      int r, px;
      if (W == 2) {
        r = id >> 1;
        px = (id & 1) ? TXC + 2 : 0;
      } else {
        r = id >> 2;
        px = (id & 3) < 2 ? (id & 3) : TXC + (id & 3);
      }
      hval[q] = id < Sh::XHALO_LANES;
      r = hval[q] ? r : 0;
      hpy[q] = r + OY;
      hpx[q] = px;
      hsrc[q] = cell_src<T>(x0 + px - 2, grid_row(y0 + r), nx, bnd);
    }
    constexpr int NYP = (D == 3) ? 4 : 0;  // y halo rows this warp fills
    CellSrc ysrc[NYP > 0 ? NYP : 1];
#pragma unroll
    for (int q = 0; q < NYP; ++q) ysrc[q] = cell_src<T>(x0 + lane * W, grid_row(y0 + (q < 2 ? q : TYC + q) - 2), nx, bnd);
    T Uh[NXP][NF], Uyh[NYP > 0 ? NYP : 1][NF];
    auto load_halo = [&](int m) {
      const int pl = plane_of(m);
#pragma unroll
      for (int q = 0; q < NXP; ++q)
        if (hval[q]) {
#pragma unroll
          for (int f = 0; f < NF; ++f) Uh[q][f] = ldg_cells<T>(Uin, f * Ni + pl, hsrc[q]);
        }
#pragma unroll
      for (int q = 0; q < NYP; ++q) {
#pragma unroll
        for (int f = 0; f < NF; ++f) Uyh[q][f] = ldg_cells<T>(Uin, f * Ni + pl, ysrc[q]);
      }
    };
    auto store_halo = [&](int b) {
      T u[NF];
#pragma unroll
      for (int q = 0; q < NXP; ++q)
        if (hval[q]) {
          prim_to_fields<T, D>(prim_of<T, D>(Uh[q], g.gm1), u);
#pragma unroll
          for (int f = 0; f < NF; ++f) sts(&sm.V[b][f][hpy[q]][hpx[q]], u[f]);
        }
#pragma unroll
      for (int q = 0; q < NYP; ++q) {
        prim_to_fields<T, D>(prim_of<T, D>(Uyh[q], g.gm1), u);
#pragma unroll
        for (int f = 0; f < NF; ++f) sts(&sm.V[b][f][q < 2 ? q : TYC + q][lane * W + 2], u[f]);
      }
    };
    // x face tasks: lane l < XTASK_LANES handles tile rows ra (first lane of T) and rb (second lane)
    const bool xtask = lane < Sh::XTASK_LANES;
    const int ra = xtask ? lane : 0;
    const int rb = (W == 2) ? min(ra + Sh::XTASK_LANES, XROWS - 1) : ra;
    auto plane_x = [&](int b, int qx) {
      T u[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = lane_pack(sm.V[b][f][ra + OY][qx], sm.V[b][f][rb + OY][qx], (T*)nullptr);
      return prim_from_fields<T, D>(u);
    };
    auto plane_y = [&](int b, int py) {
      T u[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) u[f] = lds<T>(&sm.V[b][f][py][lane * W + 2]);
      return prim_from_fields<T, D>(u);
    };

    // TMA producer: one bulk copy per field and tile row (jobs spread over the lanes), completing on the slot's mbarrier
    constexpr int NJOB = NF * XROWS, JPL = (NJOB + 31) / 32;
    constexpr int ROW_BYTES = TXC * (int)sizeof(S);
    int job_off[JPL];  // element offset of the row inside a plane + f * N
#pragma unroll
    for (int j = 0; j < JPL; ++j) {
      const int job = lane + 32 * j;
      const int f = job / XROWS, r = job - f * XROWS;
      job_off[j] = job < NJOB ? f * Ni + grid_row(y0 + r) + x0 : -1;
    }
    auto tma_plane = [&](const S* A, int m, S* dst_slot, unsigned long long* bar) {
      if constexpr (TMA == 2) {  // one instruction per plane: the box (TXC, rows, 1 plane, NF fields) of the tensor map
        if (lane == 0) {
          mbar_expect_tx(bar, NJOB * ROW_BYTES);
          const CUtensorMap* tm = (A == Uin) ? &tm_in : &tm_base;
          const int pm = map_index(m, nM, bnd);
          if constexpr (D == 3) tma_box4(dst_slot, tm, x0, y0, pm, 0, bar);
          else tma_box3(dst_slot, tm, x0, pm, 0, bar);
        }
        __syncwarp();
      } else {
        const int pl = plane_of(m);
        if (lane == 0) mbar_expect_tx(bar, NJOB * ROW_BYTES);
        __syncwarp();
#pragma unroll
        for (int j = 0; j < JPL; ++j)
          if (job_off[j] >= 0) tma_row(dst_slot + (size_t)(lane + 32 * j) * TXC, A + (job_off[j] + pl), ROW_BYTES, bar);
      }
    };
    if (TMA && use_tma) {
      if (lane == 0) {
#pragma unroll
        for (int i = 0; i < RING + 2; ++i) mbar_init(&sm.mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      }
      __syncwarp();
#pragma unroll
      for (int k = 0; k < 3; ++k) tma_plane(Uin, m0 + k, &sm.Uraw[k][0][0][0], &sm.mbar[k]);
      if (STAGE == 2) tma_plane(Ubase, m0, &sm.Ub[0][0][0][0], &sm.mbar[RING]);
    }
    load_halo(m0);
    store_halo(0);
    block_barrier();

    int b = 0;
    for (int m = m0; m < m1; ++m, b ^= 1) {
      const bool more = m + 1 < m1;
      // ---- phase A: high-side states of the cells just below the tile, low-side states of those just above
      if (TMA && use_tma && more) {  // every reader of the slots written here passed the last block barrier
        const int q = m - m0;
        tma_plane(Uin, m + 3, &sm.Uraw[(q + 3) % RING][0][0][0], &sm.mbar[(q + 3) % RING]);
        if (STAGE == 2) tma_plane(Ubase, m + 1, &sm.Ub[(q + 1) & 1][0][0][0], &sm.mbar[RING + ((q + 1) & 1)]);
      }
      if (more) load_halo(m + 1);
      P hiYlow, hiXlow;
      if constexpr (D == 3) {
        interpolate<T, D>(plane_y(b, 0), plane_y(b, 1), plane_y(b, 2), nullptr, &hiYlow);
        P lo;
        interpolate<T, D>(plane_y(b, TYC + 1), plane_y(b, TYC + 2), plane_y(b, TYC + 3), &lo, nullptr);
        T a[NF];
        prim_to_fields<T, D>(lo, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) sts(&sm.LOy[f][TYC][lane * W], a[f]);
      }
      if (xtask) {
        interpolate<T, D>(plane_x(b, 0), plane_x(b, 1), plane_x(b, 2), nullptr, &hiXlow);
        P lo;
        interpolate<T, D>(plane_x(b, TXC + 1), plane_x(b, TXC + 2), plane_x(b, TXC + 3), &lo, nullptr);
        T a[NF];
        prim_to_fields<T, D>(lo, a);
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          sm.LOx[f][ra][NWX] = lane_first(a[f]);
          if (W == 2) sm.LOx[f][rb][NWX] = lane_last(a[f]);
        }
      }
      block_barrier();
      // ---- phase B: flux through the tile's low faces (low-side state from the tile's first row / column);
      //      primitives of the next plane's x halo
      if constexpr (D == 3) {
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
      if (more) store_halo(b ^ 1);
      block_barrier();
    }
  }
  if (STAGE == 2) {
    const unsigned int nblocks = gridDim.x * gridDim.y * gridDim.z;
    block_reduce_and_finalize<S>(s_max, bad, sc, g, nblocks, 1);
  }
}

// ------------------------------------------------------------------------------------------------
// The tensor map of one state buffer: rank D + 1 (x, y[, z], field), box = (TXC, tile rows[, 1 plane], all fields).
template <class S, int D>
static bool make_state_tensor_map(CUtensorMap* tm, const S* U, const Geom<S>& g, int txc, int rows) {
  typedef CUresult (*Encode)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static Encode encode = nullptr;
  if (!encode) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess || !p)
      return false;
    encode = (Encode)p;
  }
  constexpr int R = D + 1;
  cuuint64_t dims[4], strides[3];
  cuuint32_t box[4], estr[4] = {1, 1, 1, 1};
  const cuuint64_t w = sizeof(S);
  dims[0] = g.n[0];
  box[0] = txc;
  if (D == 3) {
    dims[1] = g.n[1], dims[2] = g.n[2], dims[3] = D + 2;
    strides[0] = g.n[0] * w, strides[1] = (cuuint64_t)g.n[0] * g.n[1] * w, strides[2] = (cuuint64_t)g.N * w;
    box[1] = rows, box[2] = 1, box[3] = D + 2;
  } else {
    dims[1] = g.n[1], dims[2] = D + 2;
    strides[0] = g.n[0] * w, strides[1] = (cuuint64_t)g.N * w;
    box[1] = 1, box[2] = D + 2;
  }
  return encode(tm, sizeof(S) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, R, (void*)U, dims,
                strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <class T, int D, int RS, int STAGE, int NWX, int TY, int MINB, int TMA = 0, int RPT = 1>
static bool launch_march_shape(const scalar_t<T>* Uin, const scalar_t<T>* Ubase, scalar_t<T>* Uout,
                               const Geom<scalar_t<T>>& g, Scalars* sc, cudaStream_t stream, int depth) {
  using Sh = MarchShape<T, D, NWX, TY, TMA, RPT>;
  auto kern = k_march<T, D, RS, STAGE, NWX, TY, MINB, TMA, RPT>;
  // the opt-in to more than 48 KB of dynamic shared memory is a per-device attribute of the kernel
  static bool configured[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
  if (!configured[dev]) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(typename Sh::Smem)) != cudaSuccess)
      return false;
    configured[dev] = true;
  }
  constexpr int M = D - 1;
  dim3 grid, block(Sh::NT, 1, 1);
  grid.x = (g.n[0] + Sh::TXC - 1) / Sh::TXC;
  if (D == 3) {
    grid.y = (g.n[1] + Sh::TYC - 1) / Sh::TYC;
    grid.z = (g.n[M] + depth - 1) / depth;
    if (grid.y > 65535u || grid.z > 65535u) return false;
  } else {
    grid.y = (g.n[M] + depth - 1) / depth;
    grid.z = 1;
    if (grid.y > 65535u) return false;
  }
  CUtensorMap tm_in, tm_base;
  if constexpr (TMA == 2) {
    if (!make_state_tensor_map<scalar_t<T>, D>(&tm_in, Uin, g, Sh::TXC, Sh::XROWS) ||
        !make_state_tensor_map<scalar_t<T>, D>(&tm_base, Ubase, g, Sh::TXC, Sh::XROWS))
      return false;
  } else {
    memset(&tm_in, 0, sizeof tm_in);
    memset(&tm_base, 0, sizeof tm_base);
  }
  kern<<<grid, block, sizeof(typename Sh::Smem), stream>>>(Uin, Ubase, Uout, g, sc, depth, tm_in, tm_base);
  return true;
}

// Planes marched per block when the caller gives none: deep enough that the 4 extra planes of the prologue
// stay below ~10 % of the work, shallow enough to give every SM several blocks.
inline int march_default_depth(long long tiles_in_plane, int nM) {
  int depth = 128;
  while (depth > 8 && tiles_in_plane * ((nM + depth - 1) / depth) < 4 * device_sm_count()) depth >>= 1;
  return depth;
}

// Returns false when the marching kernel does not cover this shape (the caller falls back).
//   pack: cells per thread along x (0 = default = 1; 2 = packed f32x2, fp32 on an even n_x only: measured slower,
//         DESIGN.md §7)
//   block[0] (2-D): main warps per block (0 = default); block[1] (3-D): main warps TY (0 = default);
//   block[2] (3-D): rows per thread (0 / 1, or 2 with TY = 7)
//   arith: 1 = fp32 with the hardware reciprocal / reciprocal square root approximations (f32fast: inside north_star's
//          tolerances, not bit-equal to the oracle; default shapes only), 0 = IEEE-exact (default)
//   staging: 0 / 1 = every thread loads its own cells (LDG), 2 = TMA bulk copies of the tile rows into a shared-memory
//            ring (one cell per thread, n_x a multiple of 16 bytes, default tile shapes only), 3 = the same ring filled by
//            ONE tensor-map copy per plane (cp.async.bulk.tensor: SASS UTMALDG)
template <class Real, int D, int RS, int STAGE>
bool launch_march_stage(const Real* Uin, const Real* Ubase, Real* Uout, const Geom<Real>& g, Scalars* sc,
                        cudaStream_t stream, const int* block, int tile_depth, int pack, int staging, int arith) {
  if constexpr (D == 1) {
    return false;
  } else {
    constexpr bool can_pack = sizeof(Real) == 4;
    constexpr int minb = sizeof(Real) == 4 ? PH_MARCH_MINB : 1;  // one cell per thread in fp32: blocks per SM the register cap is set for
    const bool packed = can_pack && pack == 2 && (g.n[0] % 2 == 0);
    if (pack == 2 && !packed) return false;
    const int w = packed ? 2 : 1;
    const bool tma = staging == 2 && !packed && g.n[0] % (16 / (int)sizeof(Real)) == 0;
    const bool tma_map = staging == 3 && !packed && g.n[0] % (16 / (int)sizeof(Real)) == 0;  // tensor-map TMA
    // A knob this kernel cannot honour is "shape not covered" (false), never the plain kernel under the requested name:
    // TMA staging needs an unpacked row of whole 16-byte units and the default tile; arith = 1 exists in fp32, default
    // tile, per-thread loads, one cell per thread; a block_* this dimension does not read must be 0.
    if (staging < 0 || staging > 3 || (staging >= 2 && !(tma || tma_map))) return false;
    if (arith < 0 || arith > 1 || (arith == 1 && (!can_pack || packed || staging >= 2 || block[2] == 2))) return false;
    const int shape_knob = D == 2 ? block[0] : block[1];
    if ((staging >= 2 || arith == 1) && shape_knob > 0 && shape_knob != (D == 2 ? 4 : 7)) return false;
    if (D == 2 ? (block[1] != 0 || block[2] != 0) : (block[0] != 0 || block[2] < 0 || block[2] > 2)) return false;
    if (D == 3 && block[2] == 2 && (packed || staging >= 2 || (block[1] > 0 && block[1] != 7))) return false;
    if constexpr (D == 2) {
      int nwx = block[0] > 0 ? block[0] : 4;
      const long long tiles = (g.n[0] + nwx * 32 * w - 1) / (nwx * 32 * w);
      const int depth = tile_depth > 0 ? tile_depth : march_default_depth(tiles, g.n[1]);
#define PH_SHAPE(NWXV)                                                                                              \
  if (nwx == NWXV) {                                                                                                \
    if constexpr (can_pack)                                                                                         \
      if (packed) return launch_march_shape<f32x2, D, RS, STAGE, NWXV, 1, 1>(Uin, Ubase, Uout, g, sc, stream, depth); \
    return launch_march_shape<Real, D, RS, STAGE, NWXV, 1, minb>(Uin, Ubase, Uout, g, sc, stream, depth);           \
  }
      if constexpr (can_pack)
        if (arith == 1 && nwx == 4) return launch_march_shape<f32fast, D, RS, STAGE, 4, 1, minb>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (tma && nwx == 4) return launch_march_shape<Real, D, RS, STAGE, 4, 1, minb, 1>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (tma_map && nwx == 4) return launch_march_shape<Real, D, RS, STAGE, 4, 1, minb, 2>(Uin, Ubase, Uout, g, sc, stream, depth);
      PH_SHAPE(2) PH_SHAPE(3) PH_SHAPE(4) PH_SHAPE(7) PH_SHAPE(8)
#undef PH_SHAPE
      return false;
    } else {
      const int ty = block[1] > 0 ? block[1] : 7;  // 7 main warps + the halo warp = 256 threads
      const long long tiles = (long long)((g.n[0] + 32 * w - 1) / (32 * w)) * ((g.n[1] + ty - 1) / ty);
      const int depth = tile_depth > 0 ? tile_depth : march_default_depth(tiles, g.n[2]);
#define PH_SHAPE(TYV)                                                                                               \
  if (ty == TYV) {                                                                                                  \
    if constexpr (can_pack)                                                                                         \
      if (packed) return launch_march_shape<f32x2, D, RS, STAGE, 1, TYV, 1>(Uin, Ubase, Uout, g, sc, stream, depth);  \
    return launch_march_shape<Real, D, RS, STAGE, 1, TYV, (TYV > 8 ? 1 : minb)>(Uin, Ubase, Uout, g, sc, stream, depth);            \
  }
      if constexpr (can_pack)
        if (arith == 1 && ty == 7) return launch_march_shape<f32fast, D, RS, STAGE, 1, 7, minb>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (tma && ty == 7) return launch_march_shape<Real, D, RS, STAGE, 1, 7, minb, 1>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (tma_map && ty == 7) return launch_march_shape<Real, D, RS, STAGE, 1, 7, minb, 2>(Uin, Ubase, Uout, g, sc, stream, depth);
      if (block[2] == 2 && ty == 7 && !packed)  // two rows per thread: a 32 x 14 tile, one 256-thread block per SM
        return launch_march_shape<Real, D, RS, STAGE, 1, 7, PH_RPT2_MINB, 0, 2>(Uin, Ubase, Uout, g, sc, stream, depth);
      PH_SHAPE(4) PH_SHAPE(7) PH_SHAPE(8) PH_SHAPE(15)
#undef PH_SHAPE
      return false;
    }
  }
}

}  // namespace ph
