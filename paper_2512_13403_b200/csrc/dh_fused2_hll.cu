// dh_fused2_hll.cu — the fused z-sweep stage kernel (dh_fused2_impl.cuh) with the two-wave HLL (DH_OPT_RIEMANN = 1) flux.
#include "dh_fused2_impl.cuh"

namespace dh {
template cudaError_t launch_stage_fused2_rs<float, 1, false>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2_rs<double, 1, false>(const StageParams<double>&, int, int, cudaStream_t, bool*);
}  // namespace dh
