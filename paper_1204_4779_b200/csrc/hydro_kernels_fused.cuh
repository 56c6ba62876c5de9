// hydro_kernels_fused.cuh — the fused end of the Manifest <-> Delayed axis: one kernel per RK stage.
#pragma once
#include "hydro_control.cuh"

namespace ph {

// Returns false when the marching kernel does not cover this shape (the caller then uses k_delayed).
template <class Real, int D, int RS, int STAGE>
static bool launch_fused_stage(const Real* Uin, const Real* Ubase, Real* Uout, const Geom<Real>& g, Scalars* sc,
                               cudaStream_t stream, const int (&block)[3], int tile_depth, int cells_per_thread) {
  return false;
}

}  // namespace ph
