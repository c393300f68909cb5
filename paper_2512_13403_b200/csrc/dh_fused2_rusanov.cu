// dh_fused2_rusanov.cu — the fused z-sweep stage kernel (dh_fused2_impl.cuh) with the Rusanov / local Lax-Friedrichs (DH_OPT_RIEMANN = 2) flux.
#include "dh_fused2_impl.cuh"

namespace dh {
template cudaError_t launch_stage_fused2_rs<float, 2, false>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2_rs<double, 2, false>(const StageParams<double>&, int, int, cudaStream_t, bool*);
}  // namespace dh
