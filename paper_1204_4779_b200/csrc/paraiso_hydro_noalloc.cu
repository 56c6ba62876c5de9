// paraiso_hydro_noalloc.cu — paraiso_hydro_cfl_noalloc() of include/paraiso_hydro_noalloc.h: the CFL reduction (a0;
// PAPER.md:25, :736; R6) for callers that may not allocate.  It is k_cfl's arithmetic (prim_of, cfl_speed,
// bad_state of hydro_math.cuh / hydro_kernels_basic.cuh, cell by cell) with the reduction's working memory — per-block
// partials and the last-block ticket, which the handle path keeps in its cudaMalloc'ed control block — moved into a
// fixed array that is part of the library image.  No cudaMalloc / cudaFree / allocating library call in this file.
#include "../../include/paraiso_hydro_noalloc.h"

#include <cuda_runtime.h>

#include <cmath>
#include <mutex>

#include "../../include/paraiso_hydro.h"
#include "hydro_kernels_basic.cuh"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CELLS_PER_THREAD = 16;
constexpr long long NA_CELLS_PER_BLOCK = (long long)NA_THREADS * NA_CELLS_PER_THREAD;  // 4096
constexpr int NA_MAX_BLOCKS = 32768;
constexpr int NA_HEADER_BYTES = 256;  // the ticket sits alone in the first 256 bytes; only these are cleared per call
constexpr size_t NA_SCRATCH_BYTES = NA_HEADER_BYTES + (size_t)NA_MAX_BLOCKS * (sizeof(double) + sizeof(unsigned int));
static_assert(NA_SCRATCH_BYTES == PARAISO_NOALLOC_SCRATCH_BYTES, "header and scratch layout disagree");
static_assert(NA_CELLS_PER_BLOCK * NA_MAX_BLOCKS == PARAISO_NOALLOC_MAX_CELLS, "header and block shape disagree");

// The scratch itself.  One copy per GPU that loads this library, alive until the process ends, shared by every call on
// that GPU.  In HOST code below this name is only a handle for cudaGetSymbolAddress — it is NOT a device address, and a
// kernel handed `g_noalloc_scratch` by the host would read the wrong memory.  The host passes the looked-up pointer.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_SCRATCH_BYTES];

struct ScratchView {
  unsigned int* ticket;  // must be 0 when the kernel starts
  double* S;             // [NA_MAX_BLOCKS] partial maxima, widened to double; every block of a launch writes its own
  unsigned int* bad;     // [NA_MAX_BLOCKS] bad cells per block (<= 4096 each)
};
__host__ __device__ inline ScratchView view_of(unsigned char* base) {
  ScratchView v;
  v.ticket = (unsigned int*)base;
  v.S = (double*)(base + NA_HEADER_BYTES);
  v.bad = (unsigned int*)(base + NA_HEADER_BYTES + (size_t)NA_MAX_BLOCKS * sizeof(double));
  return v;
}

// Block b owns cells [b * 4096, (b + 1) * 4096); a thread takes every 256th of them, so a warp's loads are contiguous.
// The last block to hand in its partial (ticket) folds all of them and writes the three results.
template <class Real, int D>
__global__ void __launch_bounds__(NA_THREADS)
    k_cfl_noalloc(const Real* __restrict__ U, ph::Geom<Real> g, Real cfl, unsigned char* scratch, double* __restrict__ out) {
  using namespace ph;
  const ScratchView sv = view_of(scratch);
  __shared__ Real s_warp[NA_THREADS / 32];
  __shared__ unsigned int s_bad[NA_THREADS / 32];
  __shared__ bool s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  Real s = Real(0);
  unsigned int bad = 0;
  const long long first = blockIdx.x * NA_CELLS_PER_BLOCK + threadIdx.x;
#pragma unroll 4
  for (int k = 0; k < NA_CELLS_PER_THREAD; ++k) {
    const long long c = first + (long long)k * NA_THREADS;
    if (c < g.N) {
      Real u[D + 2], ir;
      load_fields<Real, D + 2>(U, g.N, c, u);
      const Prim<Real, D> V = prim_of<Real, D>(u, g.gm1, &ir);
      s = rmax(s, cfl_speed<Real, D>(V, ir, g.gamma, g.idr));  // fmax drops a NaN, as in k_cfl
      bad += (unsigned int)bad_state<Real, D>(V, u[D + 1]);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s = rmax(s, __shfl_xor_sync(0xffffffffu, s, o));
    bad += __shfl_xor_sync(0xffffffffu, bad, o);
  }
  if (lane == 0) {
    s_warp[warp] = s;
    s_bad[warp] = bad;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < NA_THREADS / 32; ++w) {
      s = rmax(s, s_warp[w]);
      bad += s_bad[w];
    }
    sv.S[blockIdx.x] = double(s);
    sv.bad[blockIdx.x] = bad;
    __threadfence();
    s_last = atomicAdd(sv.ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!s_last) return;

  __threadfence();
  double S = 0.0;  // widening is exact and monotone, so the max of the widened partials is the widened max
  unsigned long long nbad = 0;
  for (unsigned int b = threadIdx.x; b < gridDim.x; b += NA_THREADS) {
    S = fmax(S, ((volatile double*)sv.S)[b]);
    nbad += ((volatile unsigned int*)sv.bad)[b];
  }
  __shared__ double f_S[NA_THREADS / 32];
  __shared__ unsigned long long f_bad[NA_THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    S = fmax(S, __shfl_xor_sync(0xffffffffu, S, o));
    nbad += __shfl_xor_sync(0xffffffffu, nbad, o);
  }
  if (lane == 0) {
    f_S[warp] = S;
    f_bad[warp] = nbad;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < NA_THREADS / 32; ++w) {
      S = fmax(S, f_S[w]);
      nbad += f_bad[w];
    }
    out[0] = S;
    out[1] = double(rdiv(cfl, Real(S)));  // Real(S) is exact: S is a widened Real
    out[2] = double(nbad);
  }
}

// Device address of g_noalloc_scratch, looked up once per device with that device current.
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_ptr[NA_MAX_DEVICES] = {};

int scratch_for_current_device(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) return PARAISO_ECUDA;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) {
      cudaGetLastError();
      return PARAISO_ECUDA;
    }
    g_scratch_ptr[dev] = (unsigned char*)p;
  }
  *out = g_scratch_ptr[dev];
  return PARAISO_OK;
}

template <class Real>
ph::Geom<Real> geom_of(int dims, const int64_t* n, const double* extent, double gamma, long long N) {
  ph::Geom<Real> g;
  for (int a = 0; a < 3; ++a) {
    g.n[a] = a < dims ? int(n[a]) : 1;
    g.dr[a] = a < dims ? Real(extent[a] / double(n[a])) : Real(1);
    g.idr[a] = a < dims ? Real(double(n[a]) / extent[a]) : Real(0);
  }
  g.N = N;
  g.gamma = Real(gamma);
  g.gm1 = g.gamma - Real(1);
  g.igm1 = Real(1) / g.gm1;
  g.boundary = ph::BOUNDARY_PERIODIC;  // unused: no stencil
  g.integrator = 0;
  return g;
}

template <class Real>
void launch(int dims, unsigned int blocks, cudaStream_t st, const void* U, const ph::Geom<Real>& g, double cfl,
            unsigned char* scratch, double* out) {
  const Real* u = (const Real*)U;
  if (dims == 1)
    k_cfl_noalloc<Real, 1><<<blocks, NA_THREADS, 0, st>>>(u, g, Real(cfl), scratch, out);
  else if (dims == 2)
    k_cfl_noalloc<Real, 2><<<blocks, NA_THREADS, 0, st>>>(u, g, Real(cfl), scratch, out);
  else
    k_cfl_noalloc<Real, 3><<<blocks, NA_THREADS, 0, st>>>(u, g, Real(cfl), scratch, out);
}

}  // namespace

extern "C" int paraiso_hydro_cfl_noalloc(int dims, const int64_t* n, const double* extent, double gamma, int dtype,
                                         const void* U_dev, double cfl, void* cuda_stream, double* out_dev) {
  if (!n || !extent || !U_dev || !out_dev) return PARAISO_EINVAL;
  if (dims < 1 || dims > 3) return PARAISO_EINVAL;
  if (dtype != PARAISO_F32 && dtype != PARAISO_F64) return PARAISO_EINVAL;
  if (!(gamma > 1.0) || !std::isfinite(gamma)) return PARAISO_EINVAL;
  if (!(cfl > 0.0) || !std::isfinite(cfl)) return PARAISO_EINVAL;
  long long N = 1;
  for (int a = 0; a < dims; ++a) {
    if (n[a] < 1 || n[a] > 2147483647LL || !(extent[a] > 0.0) || !std::isfinite(extent[a])) return PARAISO_EINVAL;
    N *= n[a];  // < 2^27 * 2^31: cannot overflow
    if (N > PARAISO_NOALLOC_MAX_CELLS) return PARAISO_ETOOLARGE;  // more blocks than the built-in scratch has partials for
  }

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return PARAISO_ECUDA;  // no CPU fallback
  }
  unsigned char* scratch = nullptr;
  const int rc = scratch_for_current_device(&scratch);
  if (rc != PARAISO_OK) return rc;

  cudaStream_t st = (cudaStream_t)cuda_stream;
  // the ticket is the only part that must be zero at kernel start; partials are overwritten before they are read
  if (cudaMemsetAsync(scratch, 0, NA_HEADER_BYTES, st) != cudaSuccess) {
    cudaGetLastError();
    return PARAISO_ECUDA;
  }
  const unsigned int blocks = (unsigned int)((N + NA_CELLS_PER_BLOCK - 1) / NA_CELLS_PER_BLOCK);
  if (dtype == PARAISO_F32)
    launch<float>(dims, blocks, st, U_dev, geom_of<float>(dims, n, extent, gamma, N), cfl, scratch, out_dev);
  else
    launch<double>(dims, blocks, st, U_dev, geom_of<double>(dims, n, extent, gamma, N), cfl, scratch, out_dev);
  return cudaGetLastError() == cudaSuccess ? PARAISO_OK : PARAISO_ECUDA;
}
