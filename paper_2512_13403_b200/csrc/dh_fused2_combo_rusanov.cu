// dh_fused2_combo_rusanov.cu — the fused z-sweep stage kernel (dh_fused2_impl.cuh) with the Rusanov (DH_OPT_RIEMANN = 2) flux and the base state formed in
// the kernel (COMBO: out = wB B + wX U - frac dt D(U), the Shu-Osher stages of Heun / SSPRK3).
#include "dh_fused2_impl.cuh"

namespace dh {
template cudaError_t launch_stage_fused2_rs<float, 2, true>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused2_rs<double, 2, true>(const StageParams<double>&, int, int, cudaStream_t, bool*);
}  // namespace dh
