// dh_fused2_dispatch.cu — DH_OPT_RIEMANN and StageParams::combo -> the translation unit that holds that instantiation of the
// fused stage kernel (dh_fused2*.cu, dh_fused2_combo*.cu).  This file sees only the declaration of launch_stage_fused2_rs
// (dh_internal.cuh), so that every variant is compiled once, in its own translation unit, side by side with the others.
#include "dh_internal.cuh"

namespace dh {

template <class T>
cudaError_t launch_stage_fused2(const StageParams<T>& p, int limiter, int riemann, int sm_count, cudaStream_t s, bool* supported) {
  if (p.combo) {
    switch (riemann) {
      case 1: return launch_stage_fused2_rs<T, 1, true>(p, limiter, sm_count, s, supported);
      case 2: return launch_stage_fused2_rs<T, 2, true>(p, limiter, sm_count, s, supported);
      default: return launch_stage_fused2_rs<T, 0, true>(p, limiter, sm_count, s, supported);
    }
  }
  switch (riemann) {
    case 1: return launch_stage_fused2_rs<T, 1, false>(p, limiter, sm_count, s, supported);
    case 2: return launch_stage_fused2_rs<T, 2, false>(p, limiter, sm_count, s, supported);
    default: return launch_stage_fused2_rs<T, 0, false>(p, limiter, sm_count, s, supported);
  }
}
template cudaError_t launch_stage_fused2<float>(const StageParams<float>&, int, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2<double>(const StageParams<double>&, int, int, int, cudaStream_t, bool*);

}  // namespace dh
