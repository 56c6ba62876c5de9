// microbench.cu — measured issue cost of the instruction classes the Euler stage kernels are made of, on the
// device the library runs on (paraiso_hydro_debug_issue_cost, include/paraiso_hydro.h).  DESIGN.md §8 derives the
// ALU roofline from unit counts and clocks; this is the measurement behind its reading of the ncu captures:
// next to 16 independent FFMA per iteration, how many scheduler cycles does one more instruction of a class cost?
//   kind 0  FFMA      (FMA pipes: one issue slot)            kind 3  IADD3 + LOP3 pair (ALU pipe)
//   kind 1  FMNMX     (ALU pipe)                             kind 4  FFMA2 (packed f32x2: two FFMA results)
//   kind 2  FSETP + FSEL pair (ALU pipe)                     kind 5  DFMA  (FP64 pipe)
//                                                            kind 6  MUFU.RCP
// Many warps per scheduler, no dependencies between the measured instructions, no memory traffic.
#include <cuda_runtime.h>

#include "../../include/paraiso_hydro.h"

namespace {

constexpr int ITERS = 4096;
constexpr int BLOCKS_PER_SM = 4;  // x 256 threads = 8 warps per scheduler

template <int KIND, int NX>
__global__ void __launch_bounds__(256) k_issue(float* out, float a, float b, int c) {
  float x[16], y[16];
  int z[16];
  double d[16];
  unsigned long long p[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    x[i] = threadIdx.x + i;
    y[i] = threadIdx.x * 0.5f + i;
    z[i] = threadIdx.x + i;
    d[i] = threadIdx.x + 0.25 * i;
    asm("mov.b64 %0, {%1,%2};" : "=l"(p[i]) : "f"(x[i]), "f"(y[i]));
  }
  unsigned long long pa, pb;
  asm("mov.b64 %0, {%1,%2};" : "=l"(pa) : "f"(a), "f"(a));
  asm("mov.b64 %0, {%1,%2};" : "=l"(pb) : "f"(b), "f"(b));
#pragma unroll 1
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = __fmaf_rn(x[i], a, b);
#pragma unroll
    for (int i = 0; i < NX; ++i) {
      if (KIND == 0) y[i] = __fmaf_rn(y[i], a, b);
      if (KIND == 1) y[i] = fminf(y[i], x[i]);
      if (KIND == 2) y[i] = (x[i] > b) ? y[i] : x[i];
      if (KIND == 3) z[i] = (z[i] + c) ^ it;
      if (KIND == 4) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(pa), "l"(pb));
      if (KIND == 5) d[i] = __fma_rn(d[i], (double)a, (double)b);
      if (KIND == 6) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(y[i]));
    }
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    float lo, hi;
    asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p[i]));
    s += x[i] + y[i] + float(z[i]) + float(d[i]) + lo + hi;
  }
  out[blockIdx.x * 256 + threadIdx.x] = s;
}

// scheduler cycles per warp-iteration at the clock the kernel ran at (cycles = time * sm_clock / warps per scheduler)
template <int KIND, int NX>
cudaError_t time_kernel(float* out, int sms, double* ms_out) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = sms * BLOCKS_PER_SM;
  k_issue<KIND, NX><<<blocks, 256>>>(out, 1.0001f, 0.5f, 3);
  float best = 1e30f;
  for (int r = 0; r < 3; ++r) {
    cudaEventRecord(e0);
    k_issue<KIND, NX><<<blocks, 256>>>(out, 1.0001f, 0.5f, 3);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *ms_out = best;
  return cudaGetLastError();
}

template <int KIND>
cudaError_t measure(float* out, int sms, double* ms0, double* ms16) {
  cudaError_t e = time_kernel<KIND, 0>(out, sms, ms0);
  if (e != cudaSuccess) return e;
  return time_kernel<KIND, 16>(out, sms, ms16);
}

}  // namespace

extern "C" int paraiso_hydro_debug_issue_cost(int kind, double sm_clock_mhz, double* cycles_per_instruction,
                                              double* base_cycles_per_iteration) {
  if (kind < 0 || kind > 6 || !(sm_clock_mhz > 0) || !cycles_per_instruction) return PARAISO_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return PARAISO_ECUDA;
  float* out = nullptr;
  if (cudaMalloc(&out, size_t(sms) * BLOCKS_PER_SM * 256 * sizeof(float)) != cudaSuccess) return PARAISO_ENOMEM;
  double ms0 = 0, ms16 = 0;
  cudaError_t e = cudaSuccess;
  switch (kind) {
    case 0: e = measure<0>(out, sms, &ms0, &ms16); break;
    case 1: e = measure<1>(out, sms, &ms0, &ms16); break;
    case 2: e = measure<2>(out, sms, &ms0, &ms16); break;
    case 3: e = measure<3>(out, sms, &ms0, &ms16); break;
    case 4: e = measure<4>(out, sms, &ms0, &ms16); break;
    case 5: e = measure<5>(out, sms, &ms0, &ms16); break;
    default: e = measure<6>(out, sms, &ms0, &ms16); break;
  }
  cudaFree(out);
  if (e != cudaSuccess) return PARAISO_ECUDA;
  const double warps_per_scheduler = BLOCKS_PER_SM * 8 / 4.0;
  const double to_cycles = 1e-3 * sm_clock_mhz * 1e6 / ITERS / warps_per_scheduler;
  // 16 more source-level operations per iteration; kinds 2 and 3 are two instructions each
  const double per_op = (ms16 - ms0) * to_cycles / 16.0;
  *cycles_per_instruction = (kind == 2 || kind == 3) ? per_op / 2.0 : per_op;
  if (base_cycles_per_iteration) *base_cycles_per_iteration = ms0 * to_cycles;
  return PARAISO_OK;
}
