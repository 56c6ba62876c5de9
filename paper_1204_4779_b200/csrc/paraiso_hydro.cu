// paraiso_hydro.cu — C-ABI entry points (include/paraiso_hydro.h), handle, device buffers, variant
// dispatch and CUDA-graph replay.  Host code only orchestrates: every step of the path runs in the
// kernels of hydro_kernels_*.cuh.  No CPU fallback exists.
#include "../../include/paraiso_hydro.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "hydro_kernels_basic.cuh"
#include "hydro_kernels_fused.cuh"
#include "hydro_kernels_march.cuh"
#include "hydro_kernels_pack.cuh"
#include "hydro_kernels_small.cuh"

using namespace ph;

// the 2-D / 3-D instantiations live in fused_<dtype>_d<D>.cu
namespace ph {
#define PH_EXTERN1(REAL, DD, RS, ST)                                                                      \
  extern template bool launch_fused_stage<REAL, DD, RS, ST>(const REAL*, const REAL*, REAL*, const Geom<REAL>&, \
                                                            Scalars*, cudaStream_t, const int*, int);            \
  extern template bool launch_march_stage<REAL, DD, RS, ST>(const REAL*, const REAL*, REAL*, const Geom<REAL>&, \
                                                            Scalars*, cudaStream_t, const int*, int, int, int, int);
#define PH_EXTERN(REAL, DD)              \
  PH_EXTERN1(REAL, DD, RIEMANN_HLLC, 1)  \
  PH_EXTERN1(REAL, DD, RIEMANN_HLLC, 2)  \
  PH_EXTERN1(REAL, DD, RIEMANN_HLL, 1)   \
  PH_EXTERN1(REAL, DD, RIEMANN_HLL, 2)
PH_EXTERN(float, 2)
PH_EXTERN(float, 3)
PH_EXTERN(double, 2)
PH_EXTERN(double, 3)
#undef PH_EXTERN
#undef PH_EXTERN1
// the packed / shared-memory-window kernels live in pack_f<32|64>_d<D>.cu
#define PH_EXTERN_PACK1(REAL, DD, RS, ST)                                                                              \
  extern template bool launch_pack_stage<REAL, DD, RS, ST>(const REAL*, const REAL*, REAL*, const Geom<REAL>&, Scalars*, \
                                                           cudaStream_t, const int*, int);
#define PH_EXTERN_PACK(REAL, DD)             \
  PH_EXTERN_PACK1(REAL, DD, RIEMANN_HLLC, 1) \
  PH_EXTERN_PACK1(REAL, DD, RIEMANN_HLLC, 2) \
  PH_EXTERN_PACK1(REAL, DD, RIEMANN_HLL, 1)  \
  PH_EXTERN_PACK1(REAL, DD, RIEMANN_HLL, 2)
PH_EXTERN_PACK(float, 2)
PH_EXTERN_PACK(float, 3)
PH_EXTERN_PACK(double, 2)
PH_EXTERN_PACK(double, 3)
#undef PH_EXTERN_PACK1
// ... and with the interpolation variants other than MINBEE in pack_lim_f<32|64>_d<D>.cu
#define PH_EXTERN_LIM1(REAL, DD, RS, ST, LIM)                                                                         \
  extern template bool launch_pack_stage_lim<REAL, DD, RS, ST, LIM>(const REAL*, const REAL*, REAL*, const Geom<REAL>&, \
                                                                    Scalars*, cudaStream_t);
#define PH_EXTERN_LIM(REAL, DD)                                                                               \
  PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLLC, 1, LIMITER_NONE) PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLLC, 2, LIMITER_NONE) \
  PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLL, 1, LIMITER_NONE) PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLL, 2, LIMITER_NONE)   \
  PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLLC, 1, LIMITER_MC) PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLLC, 2, LIMITER_MC)     \
  PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLL, 1, LIMITER_MC) PH_EXTERN_LIM1(REAL, DD, RIEMANN_HLL, 2, LIMITER_MC)
PH_EXTERN_LIM(float, 2)
PH_EXTERN_LIM(float, 3)
PH_EXTERN_LIM(double, 2)
PH_EXTERN_LIM(double, 3)
#undef PH_EXTERN_LIM
#undef PH_EXTERN_LIM1
#undef PH_EXTERN_PACK
}  // namespace ph

enum { VARIANT_FUSED = 0, VARIANT_MANIFEST_FLUX = 1, VARIANT_MANIFEST_ALL = 2, VARIANT_DELAYED = 3, VARIANT_MARCH = 4,
       VARIANT_FUSED1 = 5, VARIANT_PACK = 6 };
enum { KERNEL_NONE = 0, KERNEL_MANIFEST_FLUX = 1, KERNEL_MANIFEST_ALL = 2, KERNEL_DELAYED = 3, KERNEL_MARCH = 4,
       KERNEL_FUSED1 = 5, KERNEL_PACK = 6, KERNEL_SMALL1D = 7 };

struct paraiso_hydro {
  int dims = 0, dtype = 0, nf = 0;
  int64_t n[3] = {1, 1, 1};
  int64_t N = 0;
  double extent[3] = {1, 1, 1};
  double gamma = 0;
  size_t esize = 0;

  int boundary = BOUNDARY_PERIODIC, riemann = RIEMANN_HLLC, variant = VARIANT_FUSED;
  int block[3] = {0, 0, 0};
  int tile_depth = 0, cells_per_thread = 0, use_graph = 1;
  int arith = 0;       // k_march fp32: 0 IEEE-exact division / square root, 1 hardware approximations (f32fast)
  int staging = 0;     // k_march: 0 / 1 own-cell LDG, 2 TMA bulk row copies into a shared-memory ring, 3 one tensor-map copy per plane
  int integrator = 0;  // 0 midpoint (paper) | 1 Heun
  int limiter = 0;     // 0 MINBEE (Eq. 21) | 1 none (first order) | 2 monotonized central (R22): k_pack, k_delayed
  int state_kind = 0;  // 0: set_state / get_state exchange conserved variables, 1: primitive variables

  void* U[2] = {nullptr, nullptr};  // U[0]: current state / U_base; U[1]: stage-1 result
  void* V = nullptr;                // manifest_all: primitives
  void* LO[3] = {nullptr, nullptr, nullptr};
  void* HI[3] = {nullptr, nullptr, nullptr};
  void* F[3] = {nullptr, nullptr, nullptr};   // manifest_*: face fluxes
  void* Fb[3] = {nullptr, nullptr, nullptr};  // outflow boundary faces
  void* G = nullptr;                          // prescribed ghost cells: device copy of the caller's array (first use)
  Scalars* sc = nullptr;
  cudaStream_t stream = nullptr;
  bool has_state = false;
  int64_t launches = 0;
  int kernel_used = 0;       // KERNEL_*: the stage kernel of the last launch (get_option "kernel_used")
  bool shape_error = false;  // a requested kernel / launch shape did not cover the grid

  // optional per-stage CUDA-event timing on the handle's stream (paraiso_hydro_kernel_time)
  bool timing = false;
  std::vector<cudaEvent_t> ev;  // pairs (before, after) of the stage launches not yet read back
  size_t ev_used = 0;
  double timed_ms = 0;
  int64_t timed_count = 0;

  cudaGraphExec_t graph_exec = nullptr;
  int graph_steps = 0;

  std::string err;
};

static thread_local std::string g_create_error = "no error";

static int fail(paraiso_hydro* h, int code, const std::string& msg) {
  if (h)
    h->err = msg;
  else
    g_create_error = msg;
  return code;
}

#define CUDA_TRY(h, expr)                                                                              \
  do {                                                                                                 \
    cudaError_t e_ = (expr);                                                                           \
    if (e_ != cudaSuccess)                                                                             \
      return fail(h, e_ == cudaErrorMemoryAllocation ? PARAISO_ENOMEM : PARAISO_ECUDA,                 \
                  std::string(#expr) + ": " + cudaGetErrorString(e_));                                 \
  } while (0)

template <class Real>
static Geom<Real> make_geom(const paraiso_hydro* h) {
  Geom<Real> g;
  for (int a = 0; a < 3; ++a) {
    g.n[a] = int(h->n[a]);
    g.dr[a] = a < h->dims ? Real(h->extent[a] / double(h->n[a])) : Real(1);
    g.idr[a] = a < h->dims ? Real(double(h->n[a]) / h->extent[a]) : Real(0);
  }
  g.N = h->N;
  g.gamma = Real(h->gamma);
  g.gm1 = g.gamma - Real(1);
  g.igm1 = Real(1) / g.gm1;
  g.boundary = h->boundary;
  g.integrator = h->integrator;
  return g;
}

static void free_intermediates(paraiso_hydro* h) {
  cudaFree(h->V);
  cudaFree(h->G);
  h->V = h->G = nullptr;
  for (int a = 0; a < 3; ++a) {
    cudaFree(h->LO[a]);
    cudaFree(h->HI[a]);
    cudaFree(h->F[a]);
    cudaFree(h->Fb[a]);
    h->LO[a] = h->HI[a] = h->F[a] = h->Fb[a] = nullptr;
  }
}

// Sum up and recycle the recorded event pairs (blocks until the last one has completed).
static void drain_events(paraiso_hydro* h) {
  if (h->ev_used == 0) return;
  cudaEventSynchronize(h->ev[h->ev_used - 1]);
  for (size_t i = 0; i + 1 < h->ev_used; i += 2) {
    float ms = 0;
    if (cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]) == cudaSuccess) {
      h->timed_ms += ms;
      h->timed_count += 1;
    }
  }
  h->ev_used = 0;
}

static cudaEvent_t next_event(paraiso_hydro* h) {
  if (h->ev_used == h->ev.size()) {
    if (h->ev.size() >= 4096) {
      drain_events(h);
    } else {
      cudaEvent_t e = nullptr;
      cudaEventCreate(&e);
      h->ev.push_back(e);
    }
  }
  cudaEvent_t e = h->ev[h->ev_used++];
  cudaEventRecord(e, h->stream);
  return e;
}

static void drop_graph(paraiso_hydro* h) {
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  h->graph_exec = nullptr;
}

// Manifest intermediates are allocated on first use of a Manifest variant.
static int ensure_intermediates(paraiso_hydro* h) {
  const size_t field_bytes = size_t(h->nf) * h->N * h->esize;
  if (h->variant == VARIANT_MANIFEST_ALL || h->variant == VARIANT_MANIFEST_FLUX) {
    for (int a = 0; a < h->dims; ++a) {
      if (!h->F[a]) CUDA_TRY(h, cudaMalloc(&h->F[a], field_bytes));
      if (!h->Fb[a]) CUDA_TRY(h, cudaMalloc(&h->Fb[a], size_t(h->nf) * (h->N / h->n[a]) * h->esize));
    }
  }
  if (h->variant == VARIANT_MANIFEST_ALL) {
    if (!h->V) CUDA_TRY(h, cudaMalloc(&h->V, field_bytes));
    for (int a = 0; a < h->dims; ++a) {
      if (!h->LO[a]) CUDA_TRY(h, cudaMalloc(&h->LO[a], field_bytes));
      if (!h->HI[a]) CUDA_TRY(h, cudaMalloc(&h->HI[a], field_bytes));
    }
  }
  return PARAISO_OK;
}

// ------------------------------------------------------------------------------------------------
// Stage launchers.  stage 1: U[0] -> U[1] (tau = dt/2); stage 2: U[1] (+ own-cell U[0]) -> U[0] in place.
template <class Real, int D, int RS>
struct Launch {
  static unsigned int grid1d(int64_t N, int bs) { return (unsigned int)((N + bs - 1) / bs); }
  // U_base of Eq. 23: U0 in both stages of the midpoint rule; Heun's second stage starts from U1
  template <int STAGE>
  static const Real* stage_base(const paraiso_hydro* h) {
    return (const Real*)((STAGE == 2 && h->integrator == 1) ? h->U[1] : h->U[0]);
  }

  template <int A>
  static void recon_riemann(paraiso_hydro* h, const Geom<Real>& g) {
    const int bs = 256;
    const unsigned int gs = grid1d(h->N, bs);
    k_recon<Real, D, A><<<gs, bs, 0, h->stream>>>((const Real*)h->V, (Real*)h->LO[A], (Real*)h->HI[A], g, h->sc);
    k_riemann<Real, D, A, RS>
        <<<gs, bs, 0, h->stream>>>((const Real*)h->LO[A], (const Real*)h->HI[A], (Real*)h->F[A], (Real*)h->Fb[A], g, h->sc);
    h->launches += 2;
  }
  template <int A>
  static void flux(paraiso_hydro* h, const Geom<Real>& g, const Real* Uin) {
    const int bs = 128;
    k_flux<Real, D, A, RS><<<grid1d(h->N, bs), bs, 0, h->stream>>>(Uin, (Real*)h->F[A], (Real*)h->Fb[A], g, h->sc);
    h->launches += 1;
  }

  template <int STAGE>
  static void update(paraiso_hydro* h, const Geom<Real>& g, Real* Uout) {
    FluxArrays<Real, D> fa;
    for (int a = 0; a < 3; ++a) {
      fa.F[a] = (const Real*)h->F[a];
      fa.Fb[a] = (const Real*)h->Fb[a];
    }
    const int bs = 256;
    k_update<Real, D, STAGE><<<grid1d(h->N, bs), bs, 0, h->stream>>>(stage_base<STAGE>(h), Uout, fa, g, h->sc);
    h->launches += 1;
  }

  template <int STAGE>
  static void stage(paraiso_hydro* h) {
    const Geom<Real> g = make_geom<Real>(h);
    const Real* Uin = (const Real*)(STAGE == 1 ? h->U[0] : h->U[1]);
    Real* Uout = (Real*)(STAGE == 1 ? h->U[1] : h->U[0]);
    if (h->timing) next_event(h);
    stage_kernels<STAGE>(h, g, Uin, Uout);
    if (h->timing) next_event(h);
  }

  template <int STAGE>
  static void stage_kernels(paraiso_hydro* h, const Geom<Real>& g, const Real* Uin, Real* Uout) {
    if (h->limiter != LIMITER_MINBEE && (h->variant == VARIANT_MANIFEST_ALL || h->variant == VARIANT_MANIFEST_FLUX)) {
      h->shape_error = true;  // the interpolation variants live in k_pack and k_delayed
      return;
    }
    switch (h->variant) {
      case VARIANT_MANIFEST_ALL: {
        const int bs = 256;
        k_prim<Real, D><<<grid1d(h->N, bs), bs, 0, h->stream>>>(Uin, (Real*)h->V, g, h->sc);
        h->launches += 1;
        recon_riemann<0>(h, g);
        if constexpr (D > 1) recon_riemann<1>(h, g);
        if constexpr (D > 2) recon_riemann<2>(h, g);
        update<STAGE>(h, g, Uout);
        h->kernel_used = KERNEL_MANIFEST_ALL;
        break;
      }
      case VARIANT_MANIFEST_FLUX: {
        flux<0>(h, g, Uin);
        if constexpr (D > 1) flux<1>(h, g, Uin);
        if constexpr (D > 2) flux<2>(h, g, Uin);
        update<STAGE>(h, g, Uout);
        h->kernel_used = KERNEL_MANIFEST_FLUX;
        break;
      }
      default:
        on_chip_stage<STAGE>(h, g, Uin, Uout);
    }
  }

  // The on-chip end of the Manifest <-> Delayed axis: one kernel per stage.  Which kernel runs is recorded in
  // h->kernel_used (get_option "kernel_used").  An explicitly requested kernel (variant = pack / march / fused1 /
  // delayed), or the default one with any launch-shape option set, that does not cover the grid or the shape is an
  // error (PARAISO_EINVAL from the calling entry point), not a silent fallback; only variant = fused with all-default
  // options walks down the list pack -> march -> fused1 -> delayed.
  template <int STAGE>
  static void on_chip_stage(paraiso_hydro* h, const Geom<Real>& g, const Real* Uin, Real* Uout) {
    const Real* base = stage_base<STAGE>(h);
    auto try_pack = [&]() -> bool {
      if constexpr (D >= 2) {
        if (h->cells_per_thread || h->staging || h->arith) return false;
        bool ok = false;
        if (h->limiter == LIMITER_MINBEE) {
          ok = launch_pack_stage<Real, D, RS, STAGE>(Uin, base, Uout, g, h->sc, h->stream, h->block, h->tile_depth);
        } else if (!(h->block[0] || h->block[1] || h->block[2] || h->tile_depth)) {  // default launch shape only
          ok = h->limiter == LIMITER_NONE
                   ? launch_pack_stage_lim<Real, D, RS, STAGE, LIMITER_NONE>(Uin, base, Uout, g, h->sc, h->stream)
                   : launch_pack_stage_lim<Real, D, RS, STAGE, LIMITER_MC>(Uin, base, Uout, g, h->sc, h->stream);
        }
        if (ok) h->kernel_used = KERNEL_PACK;
        return ok;
      }
      return false;
    };
    auto try_march = [&]() -> bool {
      if (h->limiter != LIMITER_MINBEE) return false;  // the interpolation variants live in k_pack and k_delayed
      if (launch_march_stage<Real, D, RS, STAGE>(Uin, base, Uout, g, h->sc, h->stream, h->block, h->tile_depth,
                                                 h->cells_per_thread, h->staging, h->arith)) {
        h->kernel_used = KERNEL_MARCH;
        return true;
      }
      return false;
    };
    auto try_fused1 = [&]() -> bool {
      if (h->limiter != LIMITER_MINBEE) return false;
      if (h->cells_per_thread == 0 && h->staging == 0 && h->arith == 0 &&
          launch_fused_stage<Real, D, RS, STAGE>(Uin, base, Uout, g, h->sc, h->stream, h->block, h->tile_depth)) {
        h->kernel_used = KERNEL_FUSED1;
        return true;
      }
      return false;
    };
    auto try_delayed = [&]() -> bool {
      const int bs = h->block[0] > 0 ? h->block[0] : 128;
      if (bs > 128 || h->block[1] || h->block[2] || h->tile_depth || h->cells_per_thread || h->staging || h->arith) return false;
      if (h->limiter == LIMITER_NONE)
        k_delayed<Real, D, RS, STAGE, LIMITER_NONE><<<grid1d(h->N, bs), bs, 0, h->stream>>>(Uin, base, Uout, g, h->sc);
      else if (h->limiter == LIMITER_MC)
        k_delayed<Real, D, RS, STAGE, LIMITER_MC><<<grid1d(h->N, bs), bs, 0, h->stream>>>(Uin, base, Uout, g, h->sc);
      else
        k_delayed<Real, D, RS, STAGE><<<grid1d(h->N, bs), bs, 0, h->stream>>>(Uin, base, Uout, g, h->sc);
      h->kernel_used = KERNEL_DELAYED;
      return true;
    };
    const bool shaped = h->block[0] || h->block[1] || h->block[2] || h->tile_depth || h->cells_per_thread || h->staging || h->arith;
    bool ok = false;
    switch (h->variant) {
      case VARIANT_PACK: ok = try_pack(); break;
      case VARIANT_MARCH: ok = try_march(); break;
      case VARIANT_FUSED1: ok = try_fused1(); break;
      case VARIANT_DELAYED: ok = try_delayed(); break;
      default: {  // VARIANT_FUSED: the fastest on-chip kernel per grid kind (profiles/r2_tune_*.txt)
        if (D == 1) {
          ok = try_delayed();
        } else {
          // the shared-memory-window kernel k_pack (fp32: packed pairs, even n_x; fp64: one cell per thread); the
          // options only k_march knows (cells_per_thread, staging, arith) select k_march
          const bool march_only = h->cells_per_thread || h->staging || h->arith;
          ok = march_only ? try_march() : (try_pack() || try_march());
        }
        if (!ok && !shaped) ok = try_march() || try_fused1() || try_delayed();
      }
    }
    if (ok)
      h->launches += 1;
    else
      h->shape_error = true;
  }

  static void step(paraiso_hydro* h) {
    stage<1>(h);
    stage<2>(h);
  }

  // 1-D grids of at most 1024 cells, default variant: `nsteps` whole steps in ONE launch (hydro_kernels_small.cuh)
  static bool small_run_covers(const paraiso_hydro* h) {
    return D == 1 && h->variant == VARIANT_FUSED && h->N <= SMALL1D_MAX && !h->timing && !h->block[0] && !h->block[1] &&
           !h->block[2] && !h->tile_depth && !h->cells_per_thread && !h->staging && !h->arith;
  }
  static void small_run(paraiso_hydro* h, int64_t nsteps) {
    if constexpr (D == 1) {
      const Geom<Real> g = make_geom<Real>(h);
      const int bs = int((h->N + 31) / 32 * 32);
      Real* U = (Real*)h->U[0];
      // at most SMALL1D_MAX_STEPS steps per launch: a launch cannot be interrupted, and the kernel carries the whole
      // time-step control in and out through *sc, so consecutive launches continue exactly where the last one stopped
      for (int64_t left = nsteps; left > 0; left -= SMALL1D_MAX_STEPS) {
        const long long k = (long long)(left < SMALL1D_MAX_STEPS ? left : SMALL1D_MAX_STEPS);
        if (h->limiter == LIMITER_NONE)
          k_small1d<Real, RS, LIMITER_NONE><<<1, bs, 0, h->stream>>>(U, g, h->sc, k);
        else if (h->limiter == LIMITER_MC)
          k_small1d<Real, RS, LIMITER_MC><<<1, bs, 0, h->stream>>>(U, g, h->sc, k);
        else
          k_small1d<Real, RS, LIMITER_MINBEE><<<1, bs, 0, h->stream>>>(U, g, h->sc, k);
        h->launches += 1;
      }
      h->kernel_used = KERNEL_SMALL1D;
    }
  }

  static void cfl(paraiso_hydro* h) {
    const Geom<Real> g = make_geom<Real>(h);
    const int bs = 256;
    int64_t blocks = (h->N + bs - 1) / bs;
    if (blocks > device_sm_count() * 8) blocks = device_sm_count() * 8;
    k_cfl<Real, D><<<(unsigned int)blocks, bs, 0, h->stream>>>((const Real*)h->U[0], g, h->sc);
    h->launches += 1;
  }

  template <bool TO_CONS>
  static void convert(paraiso_hydro* h, const void* in, void* out) {
    const int bs = 256;
    k_convert<Real, D, TO_CONS><<<grid1d(h->N, bs), bs, 0, h->stream>>>((const Real*)in, (Real*)out, make_geom<Real>(h));
    h->launches += 1;
  }

  // ghost cells of buffer U[which] := those of h->G (R23)
  static void inject(paraiso_hydro* h, int which) {
    const int bs = 256;
    k_inject_ghosts<Real, D><<<grid1d(h->N, bs), bs, 0, h->stream>>>((Real*)h->U[which], (const Real*)h->G, make_geom<Real>(h));
    h->launches += 1;
  }

  static void control(paraiso_hydro* h, int mode, double a, double b) {
    k_control<Real><<<1, 1, 0, h->stream>>>(h->sc, make_geom<Real>(h), mode, a, b);
    h->launches += 1;
  }
};

template <class F>
static void dispatch(paraiso_hydro* h, F&& f) {
#define PH_CASE(REAL, DD)                                    \
  if (h->riemann == RIEMANN_HLLC)                            \
    f(Launch<REAL, DD, RIEMANN_HLLC>{});                     \
  else                                                       \
    f(Launch<REAL, DD, RIEMANN_HLL>{});
  if (h->dtype == PARAISO_F32) {
    if (h->dims == 1) { PH_CASE(float, 1) }
    else if (h->dims == 2) { PH_CASE(float, 2) }
    else { PH_CASE(float, 3) }
  } else {
    if (h->dims == 1) { PH_CASE(double, 1) }
    else if (h->dims == 2) { PH_CASE(double, 2) }
    else { PH_CASE(double, 3) }
  }
#undef PH_CASE
}

static int check_launch(paraiso_hydro* h) {
  if (h->shape_error) {
    h->shape_error = false;
    cudaGetLastError();
    return fail(h, PARAISO_EINVAL, "the requested kernel variant / launch shape does not cover this grid (shape not covered)");
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, PARAISO_ECUDA, std::string("kernel launch: ") + cudaGetErrorString(e));
  return PARAISO_OK;
}

// ------------------------------------------------------------------------------------------------
extern "C" {

int paraiso_hydro_create(paraiso_hydro_t** out, int dims, const int64_t* n, const double* extent, double gamma,
                         int dtype) {
  if (!out || !n || !extent) return fail(nullptr, PARAISO_EINVAL, "create: null pointer");
  if (dims < 1 || dims > 3) return fail(nullptr, PARAISO_EINVAL, "create: dims must be 1, 2 or 3");
  if (dtype != PARAISO_F32 && dtype != PARAISO_F64) return fail(nullptr, PARAISO_EINVAL, "create: bad dtype");
  if (!(gamma > 1.0) || !std::isfinite(gamma)) return fail(nullptr, PARAISO_EINVAL, "create: gamma must be > 1");
  int64_t N = 1;
  for (int a = 0; a < dims; ++a) {
    if (n[a] < 4 || n[a] > (1ll << 30)) return fail(nullptr, PARAISO_EINVAL, "create: every n[a] must be >= 4");
    if (!(extent[a] > 0.0) || !std::isfinite(extent[a])) return fail(nullptr, PARAISO_EINVAL, "create: extent must be > 0");
    N *= n[a];
    if (N > (1ll << 31) / 8) return fail(nullptr, PARAISO_EINVAL, "create: grid too large (nf*N must stay below 2^31)");
  }
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0)
    return fail(nullptr, PARAISO_ECUDA,
                std::string("create: no usable CUDA device (") + cudaGetErrorString(e) + "); there is no CPU fallback");
  paraiso_hydro* h = new paraiso_hydro;
  h->dims = dims;
  h->dtype = dtype;
  h->nf = dims + 2;
  h->N = N;
  h->gamma = gamma;
  h->esize = dtype == PARAISO_F32 ? 4 : 8;
  for (int a = 0; a < dims; ++a) {
    h->n[a] = n[a];
    h->extent[a] = extent[a];
  }
  const size_t bytes = size_t(h->nf) * N * h->esize;
  for (int b = 0; b < 2; ++b) {
    e = cudaMalloc(&h->U[b], bytes);
    if (e != cudaSuccess) {
      fail(nullptr, PARAISO_ENOMEM, std::string("create: cudaMalloc(state): ") + cudaGetErrorString(e));
      paraiso_hydro_destroy(h);
      return PARAISO_ENOMEM;
    }
  }
  e = cudaMalloc((void**)&h->sc, sizeof(Scalars));
  if (e == cudaSuccess) e = cudaMemset(h->sc, 0, sizeof(Scalars));
  if (e != cudaSuccess) {
    fail(nullptr, PARAISO_ENOMEM, std::string("create: scalars: ") + cudaGetErrorString(e));
    paraiso_hydro_destroy(h);
    return PARAISO_ENOMEM;
  }
  h->err = "no error";
  *out = h;
  return PARAISO_OK;
}

int paraiso_hydro_destroy(paraiso_hydro_t* h) {
  if (!h) return PARAISO_OK;
  cudaStreamSynchronize(h->stream);
  drop_graph(h);
  free_intermediates(h);
  for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
  cudaFree(h->U[0]);
  cudaFree(h->U[1]);
  cudaFree(h->sc);
  delete h;
  return PARAISO_OK;
}

struct OptionRef {
  int* field;
  int64_t lo, hi;
};

static bool find_option(paraiso_hydro* h, const char* key, OptionRef* ref) {
  struct Opt {
    const char* key;
    OptionRef ref;
  };
  const Opt opts[] = {{"boundary", {&h->boundary, 0, 1}},
                      {"riemann", {&h->riemann, 0, 1}},
                      {"variant", {&h->variant, 0, 6}},
                      {"block_x", {&h->block[0], 0, 1024}},
                      {"block_y", {&h->block[1], 0, 1024}},
                      {"block_z", {&h->block[2], 0, 64}},
                      {"tile_depth", {&h->tile_depth, 0, 1 << 20}},
                      {"cells_per_thread", {&h->cells_per_thread, 0, 8}},
                      {"graph", {&h->use_graph, 0, 1}},
                      {"state_kind", {&h->state_kind, 0, 1}},
                      {"integrator", {&h->integrator, 0, 1}},
                      {"limiter", {&h->limiter, 0, 2}},
                      {"staging", {&h->staging, 0, 3}},
                      {"arith", {&h->arith, 0, 1}},
                      {"kernel_used", {&h->kernel_used, 0, 0}}};  // read-only: KERNEL_* of the last stage launch
  for (const Opt& o : opts)
    if (!std::strcmp(key, o.key)) {
      *ref = o.ref;
      return true;
    }
  return false;
}

int paraiso_hydro_set_option(paraiso_hydro_t* h, const char* key, int64_t value) {
  if (!h || !key) return fail(h, PARAISO_EINVAL, "set_option: null pointer");
  OptionRef r;
  if (!find_option(h, key, &r)) return fail(h, PARAISO_EINVAL, std::string("set_option: unknown key ") + key);
  if (value < r.lo || value > r.hi) return fail(h, PARAISO_EINVAL, std::string("set_option: value out of range for ") + key);
  if (*r.field != int(value)) drop_graph(h);  // a captured graph is valid only for the options it was captured with
  *r.field = int(value);
  return PARAISO_OK;
}

int paraiso_hydro_get_option(paraiso_hydro_t* h, const char* key, int64_t* value) {
  if (!h || !key || !value) return fail(h, PARAISO_EINVAL, "get_option: null pointer");
  OptionRef r;
  if (!find_option(h, key, &r)) return fail(h, PARAISO_EINVAL, std::string("get_option: unknown key ") + key);
  *value = *r.field;
  return PARAISO_OK;
}

int paraiso_hydro_set_stream(paraiso_hydro_t* h, void* cuda_stream) {
  if (!h) return fail(h, PARAISO_EINVAL, "set_stream: null handle");
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  h->stream = (cudaStream_t)cuda_stream;
  drop_graph(h);
  return PARAISO_OK;
}

int paraiso_hydro_set_state(paraiso_hydro_t* h, const void* U) {
  if (!h || !U) return fail(h, PARAISO_EINVAL, "set_state: null pointer");
  const size_t bytes = size_t(h->nf) * h->N * h->esize;
  CUDA_TRY(h, cudaMemcpyAsync(h->U[0], U, bytes, cudaMemcpyDefault, h->stream));
  dispatch(h, [&](auto L) {
    if (h->state_kind == 1) L.template convert<true>(h, h->U[0], h->U[0]);
    L.control(h, CTRL_RESET, 0, 0);
    L.cfl(h);
  });
  h->has_state = true;
  return check_launch(h);
}

int paraiso_hydro_get_state(paraiso_hydro_t* h, void* U_out) {
  if (!h || !U_out) return fail(h, PARAISO_EINVAL, "get_state: null pointer");
  if (!h->has_state) return fail(h, PARAISO_ESTATE, "get_state: no state set");
  const size_t bytes = size_t(h->nf) * h->N * h->esize;
  const void* src = h->U[0];
  if (h->state_kind == 1) {  // primitives are formed in the stage buffer, which is free between steps
    dispatch(h, [&](auto L) { L.template convert<false>(h, h->U[0], h->U[1]); });
    src = h->U[1];
  }
  CUDA_TRY(h, cudaMemcpyAsync(U_out, src, bytes, cudaMemcpyDefault, h->stream));
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, U_out);
  if (e != cudaSuccess || at.type == cudaMemoryTypeUnregistered || at.type == cudaMemoryTypeHost) {
    cudaGetLastError();
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  }
  return PARAISO_OK;
}

int paraiso_hydro_cfl_dt(paraiso_hydro_t* h, double cfl, double* dt_out) {
  if (!h || !dt_out) return fail(h, PARAISO_EINVAL, "cfl_dt: null pointer");
  if (!(cfl > 0.0) || !std::isfinite(cfl)) return fail(h, PARAISO_EINVAL, "cfl_dt: cfl must be finite and > 0");
  if (!h->has_state) return fail(h, PARAISO_ESTATE, "cfl_dt: no state set");
  double S = 0;
  CUDA_TRY(h, cudaMemcpyAsync(&S, &h->sc->S_last, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  // same IEEE division, in the handle's precision, that the device finaliser performs
  *dt_out = h->dtype == PARAISO_F32 ? double(float(cfl) / float(S)) : cfl / S;
  return PARAISO_OK;
}

int paraiso_hydro_step(paraiso_hydro_t* h, double dt) {
  if (!h) return fail(h, PARAISO_EINVAL, "step: null handle");
  if (!h->has_state) return fail(h, PARAISO_ESTATE, "step: no state set");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, PARAISO_EINVAL, "step: dt must be finite and > 0");
  int rc = ensure_intermediates(h);
  if (rc) return rc;
  dispatch(h, [&](auto L) {
    L.control(h, CTRL_MANUAL_DT, dt, 0);
    if (L.small_run_covers(h))
      L.small_run(h, 1);
    else
      L.step(h);
  });
  return check_launch(h);
}

// Brings the caller's ghost array (host or device) into the handle's device copy.
static int stage_ghosts(paraiso_hydro* h, const void* G) {
  const size_t bytes = size_t(h->nf) * h->N * h->esize;
  if (!h->G) CUDA_TRY(h, cudaMalloc(&h->G, bytes));
  CUDA_TRY(h, cudaMemcpyAsync(h->G, G, bytes, cudaMemcpyDefault, h->stream));
  return PARAISO_OK;
}

int paraiso_hydro_set_ghosts(paraiso_hydro_t* h, const void* G) {
  if (!h || !G) return fail(h, PARAISO_EINVAL, "set_ghosts: null pointer");
  if (!h->has_state) return fail(h, PARAISO_ESTATE, "set_ghosts: no state set");
  int rc = stage_ghosts(h, G);
  if (rc) return rc;
  dispatch(h, [&](auto L) { L.inject(h, 0); });
  return check_launch(h);
}

int paraiso_hydro_step_ghosts(paraiso_hydro_t* h, double dt, const void* G_mid) {
  if (!h || !G_mid) return fail(h, PARAISO_EINVAL, "step_ghosts: null pointer");
  if (!h->has_state) return fail(h, PARAISO_ESTATE, "step_ghosts: no state set");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, PARAISO_EINVAL, "step_ghosts: dt must be finite and > 0");
  int rc = ensure_intermediates(h);
  if (rc) return rc;
  rc = stage_ghosts(h, G_mid);
  if (rc) return rc;
  dispatch(h, [&](auto L) {
    L.control(h, CTRL_MANUAL_DT, dt, 0);
    L.template stage<1>(h);
    L.inject(h, 1);
    L.template stage<2>(h);
  });
  return check_launch(h);
}

// Captures `nsteps` device-paced steps into a graph (kernels read dt and lambda from the scalar block, so the
// same graph is valid for every step).
static int capture_graph(paraiso_hydro* h, int nsteps) {
  drop_graph(h);
  cudaStream_t cap;
  CUDA_TRY(h, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
  cudaStream_t user = h->stream;
  h->stream = cap;
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
  const int64_t before = h->launches;
  if (e == cudaSuccess) {
    dispatch(h, [&](auto L) {
      for (int s = 0; s < nsteps; ++s) L.step(h);
    });
    e = cudaStreamEndCapture(cap, &graph);
  }
  h->launches = before;
  h->stream = user;
  if (h->shape_error) {
    if (graph) cudaGraphDestroy(graph);
    cudaStreamDestroy(cap);
    return check_launch(h);
  }
  if (e == cudaSuccess) e = cudaGraphInstantiate(&h->graph_exec, graph, 0);
  if (graph) cudaGraphDestroy(graph);
  cudaStreamDestroy(cap);
  if (e != cudaSuccess) {
    h->graph_exec = nullptr;
    return fail(h, PARAISO_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e));
  }
  h->graph_steps = nsteps;
  return PARAISO_OK;
}

static int64_t launches_per_step(const paraiso_hydro* h) {
  switch (h->variant) {
    case VARIANT_MANIFEST_ALL: return 2 * (2 + 2 * h->dims);
    case VARIANT_MANIFEST_FLUX: return 2 * (1 + h->dims);
    default: return 2;
  }
}

static int enqueue_steps(paraiso_hydro* h, int64_t nsteps) {
  bool small = false;
  dispatch(h, [&](auto L) { small = L.small_run_covers(h); });
  if (small) {  // the whole chunk of steps in one launch
    if (nsteps > 0) dispatch(h, [&](auto L) { L.small_run(h, nsteps); });
    return check_launch(h);
  }
  const int chunk = 8;  // steps per graph
  int64_t left = nsteps;
  if (h->use_graph && !h->timing && nsteps >= chunk) {
    if (!h->graph_exec || h->graph_steps != chunk) {
      int rc = capture_graph(h, chunk);
      if (rc) return rc;
    }
    while (left >= chunk) {
      CUDA_TRY(h, cudaGraphLaunch(h->graph_exec, h->stream));
      h->launches += chunk * launches_per_step(h);
      left -= chunk;
    }
  }
  if (left > 0)
    dispatch(h, [&](auto L) {
      for (int64_t s = 0; s < left; ++s) L.step(h);
    });
  return check_launch(h);
}

int paraiso_hydro_run(paraiso_hydro_t* h, double cfl, int64_t nsteps, double t_end, int64_t* steps_done,
                      double* t_out) {
  if (!h) return fail(h, PARAISO_EINVAL, "run: null handle");
  if (!h->has_state) return fail(h, PARAISO_ESTATE, "run: no state set");
  if (!(cfl > 0.0) || !std::isfinite(cfl) || nsteps < 0) return fail(h, PARAISO_EINVAL, "run: bad cfl or nsteps");
  int rc = ensure_intermediates(h);
  if (rc) return rc;
  dispatch(h, [&](auto L) { L.control(h, CTRL_BEGIN_RUN, cfl, t_end > 0.0 ? t_end : 0.0); });
  if (!(t_end > 0.0)) {
    rc = enqueue_steps(h, nsteps);
    if (rc) return rc;
    if (steps_done) *steps_done = nsteps;
    return PARAISO_OK;
  }
  // t_end given: enqueue in chunks and look at the device clock between them; kernels of steps beyond
  // t_end return immediately (Scalars::done).
  struct {
    double t;
    long long steps;
    int done;
  } st = {0, 0, 0};
  long long steps0 = 0;
  CUDA_TRY(h, cudaMemcpyAsync(&steps0, &h->sc->steps, sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaMemcpyAsync(&st.t, &h->sc->t, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  st.steps = steps0;  // nsteps == 0: nothing runs, report the current clock
  int64_t issued = 0;
  while (issued < nsteps) {
    const int64_t c = std::min<int64_t>(64, nsteps - issued);
    rc = enqueue_steps(h, c);
    if (rc) return rc;
    issued += c;
    CUDA_TRY(h, cudaMemcpyAsync(&st.t, &h->sc->t, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(&st.steps, &h->sc->steps, sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(&st.done, &h->sc->done, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (st.done) break;
  }
  if (steps_done) *steps_done = st.steps - steps0;
  if (t_out) *t_out = st.t;
  return PARAISO_OK;
}

int paraiso_hydro_sync(paraiso_hydro_t* h) {
  if (!h) return fail(h, PARAISO_EINVAL, "sync: null handle");
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  return PARAISO_OK;
}

int paraiso_hydro_time(paraiso_hydro_t* h, double* t_out, int64_t* steps_out) {
  if (!h) return fail(h, PARAISO_EINVAL, "time: null handle");
  double t = 0;
  long long s = 0;
  CUDA_TRY(h, cudaMemcpyAsync(&t, &h->sc->t, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaMemcpyAsync(&s, &h->sc->steps, sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  if (t_out) *t_out = t;
  if (steps_out) *steps_out = s;
  return PARAISO_OK;
}

int paraiso_hydro_stats(paraiso_hydro_t* h, int64_t* nonfinite_cells) {
  if (!h) return fail(h, PARAISO_EINVAL, "stats: null handle");
  long long nf = 0;
  CUDA_TRY(h, cudaMemcpyAsync(&nf, &h->sc->nonfinite, sizeof(long long), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(h, cudaStreamSynchronize(h->stream));
  if (nonfinite_cells) *nonfinite_cells = nf;
  if (nf > 0) return fail(h, PARAISO_ENONFINITE, "stats: non-finite or non-positive rho/p encountered");
  return PARAISO_OK;
}

int paraiso_hydro_launch_count(paraiso_hydro_t* h, int64_t* launches) {
  if (!h || !launches) return fail(h, PARAISO_EINVAL, "launch_count: null pointer");
  *launches = h->launches;
  return PARAISO_OK;
}

int paraiso_hydro_kernel_time(paraiso_hydro_t* h, int enable, double* total_ms, int64_t* stage_launches) {
  if (!h) return fail(h, PARAISO_EINVAL, "kernel_time: null handle");
  if (enable >= 0) {
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    h->ev_used = 0;
    h->timed_ms = 0;
    h->timed_count = 0;
    h->timing = enable != 0;
  } else {
    drain_events(h);
  }
  if (total_ms) *total_ms = h->timed_ms;
  if (stage_launches) *stage_launches = h->timed_count;
  return PARAISO_OK;
}

const char* paraiso_hydro_last_error(const paraiso_hydro_t* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

const char* paraiso_hydro_version(void) { return "paraiso_hydro 0.1 sm_100a"; }

}  // extern "C"
