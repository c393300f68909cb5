// dh_fused2.cu — the fused z-sweep stage kernel (dh_fused2_impl.cuh) with the HLLC (DH_OPT_RIEMANN = 0, default) flux.
#include "dh_fused2_impl.cuh"

namespace dh {
template cudaError_t launch_stage_fused2_rs<float, 0>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2_rs<double, 0>(const StageParams<double>&, int, int, cudaStream_t, bool*);

// DH_OPT_RIEMANN -> the translation unit that holds that flux
template <class T>
cudaError_t launch_stage_fused2(const StageParams<T>& p, int limiter, int riemann, int sm_count, cudaStream_t s, bool* supported) {
  switch (riemann) {
    case 1: return launch_stage_fused2_rs<T, 1>(p, limiter, sm_count, s, supported);
    case 2: return launch_stage_fused2_rs<T, 2>(p, limiter, sm_count, s, supported);
    default: return launch_stage_fused2_rs<T, 0>(p, limiter, sm_count, s, supported);
  }
}
template cudaError_t launch_stage_fused2<float>(const StageParams<float>&, int, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2<double>(const StageParams<double>&, int, int, int, cudaStream_t, bool*);
}  // namespace dh
