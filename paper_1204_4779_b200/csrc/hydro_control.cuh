// hydro_control.cuh — device-resident time-step control: the CFL max reduction (warp shuffle ->
// block -> one atomicMax per block), the "last block done" finaliser that turns S into the next
// dt and the stage coefficients lambda_a = tau / dr_a without a host round trip, and the 1-thread
// control kernel the host uses to set a manual dt or to start a device-paced run.
// PAPER.md:25, 736 (CFL condition), OM Reduce/Broadcast semantics PAPER.md:180-197; R6, R18.
#pragma once
#include "hydro_math.cuh"

namespace ph {

// One block of scalars per handle, in device memory.  Reals are stored widened to double (exact).
struct Scalars {
  unsigned long long S_bits;  // running max of s over the cells of the state being produced (Real bit pattern)
  unsigned int ticket;        // blocks that have finished the reducing kernel in flight
  int last;                   // the step in flight lands on t_end
  int done;                   // t_end reached: further stage kernels return immediately
  int auto_dt;                // 1: finaliser derives the next dt from S (run); 0: host sets dt (step)
  double t, t_end, cfl;
  long long steps;
  long long nonfinite;
  double S_last;              // S of the current state
  double dt;                  // dt of the step in flight / of the next step
  double lam[2][3];           // lambda_a for stage 1 (tau = dt/2) and stage 2 (tau = dt)
};

template <class Real>
__device__ __forceinline__ unsigned long long real_bits(Real x);
template <>
__device__ __forceinline__ unsigned long long real_bits<float>(float x) {
  return (unsigned long long)__float_as_uint(x);
}
template <>
__device__ __forceinline__ unsigned long long real_bits<double>(double x) {
  return (unsigned long long)__double_as_longlong(x);
}
template <class Real>
__device__ __forceinline__ Real bits_real(unsigned long long b);
template <>
__device__ __forceinline__ float bits_real<float>(unsigned long long b) {
  return __uint_as_float((unsigned int)b);
}
template <>
__device__ __forceinline__ double bits_real<double>(unsigned long long b) {
  return __longlong_as_double((long long)b);
}

// lambda_a = tau / dr_a for both stages (DESIGN.md §4 "stage")
template <class Real>
__device__ __forceinline__ void set_lambdas(Scalars* sc, Real dt, const Geom<Real>& g) {
  sc->dt = double(dt);
  const Real tau1 = g.integrator == 1 ? dt : Real(0.5) * dt;  // Heun: both stages advance by dt
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    sc->lam[0][a] = double(rdiv(tau1, g.dr[a]));
    sc->lam[1][a] = double(rdiv(dt, g.dr[a]));
  }
}

// dt of the next step from S of the current state; clamps the last step onto t_end (R18)
template <class Real>
__device__ __forceinline__ void plan_next_step(Scalars* sc, const Geom<Real>& g) {
  if (sc->t_end > 0.0 && sc->t >= sc->t_end) {
    sc->done = 1;
    return;
  }
  Real dt = rdiv(Real(sc->cfl), Real(sc->S_last));
  sc->last = 0;
  if (sc->t_end > 0.0 && sc->t + double(dt) >= sc->t_end) {
    dt = Real(sc->t_end - sc->t);
    sc->last = 1;
  }
  set_lambdas(sc, dt, g);
}

// Called by every thread of a reducing kernel (all threads of the block must call it).
//   s    this thread's max of (|v_a|+c)/dr_a over its cells (0 if none)
//   bad  number of this thread's cells with non-finite or non-positive rho / p
//   advance  1 when the kernel completes a time step (last stage), 0 for the standalone reduction
template <class Real>
__device__ __forceinline__ void block_reduce_and_finalize(Real s, int bad, Scalars* sc, const Geom<Real>& g,
                                                          unsigned int nblocks, int advance) {
  __shared__ Real s_warp[32];
  __shared__ int s_bad[32];
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int nthreads = blockDim.x * blockDim.y * blockDim.z;
  const int lane = tid & 31, warp = tid >> 5;
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
  if (warp == 0) {
    const int nw = (nthreads + 31) >> 5;
    s = lane < nw ? s_warp[lane] : Real(0);
    bad = lane < nw ? s_bad[lane] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s = rmax(s, __shfl_xor_sync(0xffffffffu, s, o));
      bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if (lane == 0) {
      // non-negative IEEE values order like their bit patterns; a NaN never raises the max (fmax drops it)
      if (s > Real(0)) atomicMax(&sc->S_bits, real_bits(s));
      if (bad) atomicAdd((unsigned long long*)&sc->nonfinite, (unsigned long long)bad);
      __threadfence();
      const unsigned int t = atomicInc(&sc->ticket, nblocks - 1);  // wraps to 0 after the last block
      if (t == nblocks - 1) {
        __threadfence();
        const unsigned long long bits = atomicExch(&sc->S_bits, 0ull);
        sc->S_last = double(bits_real<Real>(bits));
        if (advance) {
          sc->t = sc->last ? sc->t_end : sc->t + sc->dt;
          sc->steps += 1;
        }
        if (sc->auto_dt) plan_next_step(sc, g);
      }
    }
  }
}

// SMs of the current device (host side; cached per device): what the launch heuristics size their grids against.
// Falls back to the B200's 148 only if the attribute cannot be read.
inline int device_sm_count() {
  static int sms[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  if (!sms[dev]) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v < 1) return 148;
    sms[dev] = v;
  }
  return sms[dev];
}

enum { CTRL_MANUAL_DT = 0, CTRL_BEGIN_RUN = 1, CTRL_RESET = 2 };

// <<<1,1>>> host-driven control.
template <class Real>
__global__ void k_control(Scalars* sc, Geom<Real> g, int mode, double a, double b) {
  if (mode == CTRL_RESET) {  // after set_state: t = 0
    sc->S_bits = 0;
    sc->ticket = 0;
    sc->last = 0;
    sc->done = 0;
    sc->auto_dt = 0;
    sc->t = 0.0;
    sc->t_end = 0.0;
    sc->cfl = 0.0;
    sc->steps = 0;
    sc->nonfinite = 0;
  } else if (mode == CTRL_MANUAL_DT) {  // step(dt): a = dt
    sc->auto_dt = 0;
    sc->done = 0;
    sc->last = 0;
    sc->t_end = 0.0;
    set_lambdas(sc, Real(a), g);
  } else {  // run(cfl = a, t_end = b)
    sc->auto_dt = 1;
    sc->done = 0;
    sc->cfl = a;
    sc->t_end = b;
    plan_next_step(sc, g);
  }
}

}  // namespace ph
