// pack_lim_f32_d3.cu — explicit instantiations of k_pack (hydro_kernels_pack.cuh) with the interpolation variants other
// than MINBEE (R22), float, D = 3: a translation unit of its own so that the build compiles them in parallel.
#include "hydro_kernels_pack.cuh"

namespace ph {
#define PH_INST(RS, STAGE, LIM)                                                                                        \
  template bool launch_pack_stage_lim<float, 3, RS, STAGE, LIM>(const float*, const float*, float*, const Geom<float>&, \
                                                                Scalars*, cudaStream_t);
#define PH_INST4(LIM)            \
  PH_INST(RIEMANN_HLLC, 1, LIM) \
  PH_INST(RIEMANN_HLLC, 2, LIM) \
  PH_INST(RIEMANN_HLL, 1, LIM)  \
  PH_INST(RIEMANN_HLL, 2, LIM)
PH_INST4(LIMITER_NONE)
PH_INST4(LIMITER_MC)
#undef PH_INST4
#undef PH_INST
}  // namespace ph
