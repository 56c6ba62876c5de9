// paraiso_wave.cu — the paper's linear-wave example (§2.3, Table 2) behind include/paraiso_wave.h: one fused
// kernel per step (Eq. 6, Eq. 7 and the Reduce Sum of Eq. 8).  No code shared with oracle/wave_oracle.cpp.
#include "../../include/paraiso_wave.h"

#include <cuda_runtime.h>

#include <vector>

#include "../../include/paraiso_hydro.h"

namespace {

constexpr int WAVE_BLOCK = 256;

// f1 of a cell, recomputed wherever it is needed (the shifted operands of Eq. 7: "Delayed", Fig. 6)
__device__ __forceinline__ double f1_of(const double* __restrict__ f0, const double* __restrict__ g0, long long i, double dt) {
  return __dadd_rn(__ldg(f0 + i), __dmul_rn(dt, __ldg(g0 + i)));
}

__global__ void __launch_bounds__(WAVE_BLOCK)
    k_wave_step(const double* __restrict__ f0, const double* __restrict__ g0, double* __restrict__ f1o, double* __restrict__ g1o,
                long long n, double dt, double k, double c2, double two_dx, double dx, double* __restrict__ partial,
                unsigned int* ticket, double* energy) {
  const long long i = blockIdx.x * (long long)WAVE_BLOCK + threadIdx.x;
  double e = 0.0;
  if (i < n) {
    const long long ip = i + 1 == n ? 0 : i + 1, im = i == 0 ? n - 1 : i - 1;
    const double f1 = f1_of(f0, g0, i, dt), fR = f1_of(f0, g0, ip, dt), fL = f1_of(f0, g0, im, dt);
    const double g0i = __ldg(g0 + i);
    const double g1 = __dadd_rn(g0i, __dmul_rn(k, __dadd_rn(__dadd_rn(fL, fR), -__dmul_rn(2.0, f1))));
    f1o[i] = f1;
    g1o[i] = g1;
    const double dfdx = __ddiv_rn(__dadd_rn(fR, -fL), two_dx);
    const double gm = __ddiv_rn(__dadd_rn(g0i, g1), 2.0);
    e = __dmul_rn(__dmul_rn(0.5, __dadd_rn(__dmul_rn(c2, __dmul_rn(dfdx, dfdx)), __dmul_rn(gm, gm))), dx);
  }
  // Reduce Sum: lanes by butterfly, warps through shared memory in warp order, blocks in block order by the last block
  __shared__ double s_warp[WAVE_BLOCK / 32];
  __shared__ bool last;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = e;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < WAVE_BLOCK / 32; ++w) s += s_warp[w];
    partial[blockIdx.x] = s;
    __threadfence();
    last = atomicInc(ticket, gridDim.x - 1) == gridDim.x - 1;
  }
  __syncthreads();
  if (last && threadIdx.x < 32) {
    __threadfence();
    // fixed order: lane l adds partial[l], partial[l + 32], ...; then the butterfly
    double s = 0.0;
    for (unsigned int b = threadIdx.x; b < gridDim.x; b += 32) s += ((volatile double*)partial)[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) *energy = s;
  }
}

}  // namespace

struct paraiso_wave {
  long long n = 0;
  double c = 0, dx = 0, dt = 0;
  double* f[2] = {nullptr, nullptr};
  double* g[2] = {nullptr, nullptr};
  double* partial = nullptr;
  double* energy = nullptr;  // nsteps-sized device array, grown on demand
  long long energy_cap = 0;
  unsigned int* ticket = nullptr;
  int cur = 0;
  long long launches = 0;
};

extern "C" {

int paraiso_wave_create(paraiso_wave_t** out, int64_t n, double c) {
  if (!out || n < 3 || n > (1ll << 40) || !(c > 0.0)) return PARAISO_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return PARAISO_ECUDA;  // no CPU fallback
  paraiso_wave* h = new paraiso_wave;
  h->n = n;
  h->c = c;
  h->dx = 2.0 * 3.14159265358979323846 / double(n);
  h->dt = h->dx / c;
  const long long blocks = (n + WAVE_BLOCK - 1) / WAVE_BLOCK;
  bool ok = true;
  for (int b = 0; b < 2; ++b) {
    ok = ok && cudaMalloc(&h->f[b], n * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->g[b], n * sizeof(double)) == cudaSuccess;
  }
  ok = ok && cudaMalloc(&h->partial, blocks * sizeof(double)) == cudaSuccess;
  ok = ok && cudaMalloc(&h->ticket, sizeof(unsigned int)) == cudaSuccess;
  ok = ok && cudaMemset(h->ticket, 0, sizeof(unsigned int)) == cudaSuccess;
  if (!ok) {
    paraiso_wave_destroy(h);
    return PARAISO_ENOMEM;
  }
  *out = h;
  return PARAISO_OK;
}

int paraiso_wave_destroy(paraiso_wave_t* h) {
  if (!h) return PARAISO_OK;
  cudaDeviceSynchronize();
  for (int b = 0; b < 2; ++b) {
    cudaFree(h->f[b]);
    cudaFree(h->g[b]);
  }
  cudaFree(h->partial);
  cudaFree(h->energy);
  cudaFree(h->ticket);
  delete h;
  return PARAISO_OK;
}

int paraiso_wave_set_state(paraiso_wave_t* h, const double* f, const double* g) {
  if (!h || !f || !g) return PARAISO_EINVAL;
  if (cudaMemcpy(h->f[h->cur], f, h->n * sizeof(double), cudaMemcpyDefault) != cudaSuccess) return PARAISO_ECUDA;
  if (cudaMemcpy(h->g[h->cur], g, h->n * sizeof(double), cudaMemcpyDefault) != cudaSuccess) return PARAISO_ECUDA;
  return PARAISO_OK;
}

int paraiso_wave_get_state(paraiso_wave_t* h, double* f_out, double* g_out) {
  if (!h || !f_out || !g_out) return PARAISO_EINVAL;
  if (cudaMemcpy(f_out, h->f[h->cur], h->n * sizeof(double), cudaMemcpyDefault) != cudaSuccess) return PARAISO_ECUDA;
  if (cudaMemcpy(g_out, h->g[h->cur], h->n * sizeof(double), cudaMemcpyDefault) != cudaSuccess) return PARAISO_ECUDA;
  return PARAISO_OK;
}

int paraiso_wave_step(paraiso_wave_t* h, int64_t nsteps, double* energy_out) {
  if (!h || nsteps < 0) return PARAISO_EINVAL;
  if (nsteps == 0) return PARAISO_OK;
  if (nsteps > h->energy_cap) {
    cudaFree(h->energy);
    h->energy = nullptr;
    if (cudaMalloc(&h->energy, nsteps * sizeof(double)) != cudaSuccess) return PARAISO_ENOMEM;
    h->energy_cap = nsteps;
  }
  const unsigned int blocks = (unsigned int)((h->n + WAVE_BLOCK - 1) / WAVE_BLOCK);
  const double k = h->dt * (h->c * h->c) / (h->dx * h->dx);
  for (int64_t s = 0; s < nsteps; ++s) {
    const int a = h->cur, b = a ^ 1;
    k_wave_step<<<blocks, WAVE_BLOCK>>>(h->f[a], h->g[a], h->f[b], h->g[b], h->n, h->dt, k, h->c * h->c, 2.0 * h->dx, h->dx,
                                        h->partial, h->ticket, h->energy + s);
    h->cur = b;
    h->launches += 1;
  }
  if (cudaGetLastError() != cudaSuccess) return PARAISO_ECUDA;
  if (energy_out) {
    if (cudaMemcpy(energy_out, h->energy, nsteps * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) return PARAISO_ECUDA;
  } else if (cudaDeviceSynchronize() != cudaSuccess) {
    return PARAISO_ECUDA;
  }
  return PARAISO_OK;
}

int paraiso_wave_launch_count(paraiso_wave_t* h, int64_t* launches) {
  if (!h || !launches) return PARAISO_EINVAL;
  *launches = h->launches;
  return PARAISO_OK;
}

}  // extern "C"
