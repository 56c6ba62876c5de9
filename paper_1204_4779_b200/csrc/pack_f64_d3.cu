// pack_f64_d3.cu — explicit instantiations of the packed marching stage kernels (hydro_kernels_pack.cuh) for
// fp64, D = 3: a translation unit of its own so that the build compiles the variants in parallel.
#include "hydro_kernels_pack.cuh"

namespace ph {
#define PH_INST(RS, STAGE)                                                                                       \
  template bool launch_pack_stage<double, 3, RS, STAGE>(const double*, const double*, double*, const Geom<double>&, Scalars*, \
                                                cudaStream_t, const int*, int);
PH_INST(RIEMANN_HLLC, 1)
PH_INST(RIEMANN_HLLC, 2)
PH_INST(RIEMANN_HLL, 1)
PH_INST(RIEMANN_HLL, 2)
#undef PH_INST
}  // namespace ph
