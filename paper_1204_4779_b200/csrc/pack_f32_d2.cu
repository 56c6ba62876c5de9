// pack_f32_d2.cu — explicit instantiations of the packed marching stage kernels (hydro_kernels_pack.cuh) for
// fp32, D = 2: a translation unit of its own so that the build compiles the variants in parallel.
#include "hydro_kernels_pack.cuh"

namespace ph {
#define PH_INST(RS, STAGE)                                                                                       \
  template bool launch_pack_stage<float, 2, RS, STAGE>(const float*, const float*, float*, const Geom<float>&, Scalars*, \
                                                cudaStream_t, const int*, int);
PH_INST(RIEMANN_HLLC, 1)
PH_INST(RIEMANN_HLLC, 2)
PH_INST(RIEMANN_HLL, 1)
PH_INST(RIEMANN_HLL, 2)
#undef PH_INST
}  // namespace ph
