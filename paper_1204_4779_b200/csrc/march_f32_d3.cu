// march_f32_d3.cu — explicit instantiations of the marching stage kernels (hydro_kernels_march.cuh) for
// Real = float, D = 3: a translation unit of its own so that the build compiles the variants in parallel.
#include "hydro_kernels_march.cuh"

namespace ph {
#define PH_INST(RS, STAGE)                                                                                         \
  template bool launch_march_stage<float, 3, RS, STAGE>(const float*, const float*, float*, const Geom<float>&, \
                                                          Scalars*, cudaStream_t, const int*, int, int, int, int);
PH_INST(RIEMANN_HLLC, 1)
PH_INST(RIEMANN_HLLC, 2)
PH_INST(RIEMANN_HLL, 1)
PH_INST(RIEMANN_HLL, 2)
#undef PH_INST
}  // namespace ph
