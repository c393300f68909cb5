// dh_fused2.cu — the fused z-sweep stage kernel (dh_fused2_impl.cuh) with the HLLC (DH_OPT_RIEMANN = 0, default) flux.
#include "dh_fused2_impl.cuh"

namespace dh {
template cudaError_t launch_stage_fused2_rs<float, 0, false>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2_rs<double, 0, false>(const StageParams<double>&, int, int, cudaStream_t, bool*);
}  // namespace dh
