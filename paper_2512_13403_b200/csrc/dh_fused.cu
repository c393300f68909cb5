// dh_fused.cu — fused z-sweep stage kernel (placeholder until the kernel lands: reports "unsupported"
// so that dh_step uses the gather kernels).
#include "dh_internal.cuh"

namespace dh {

template <class T>
cudaError_t launch_stage_fused(const StageParams<T>&, int, int, cudaStream_t, bool* supported) {
  *supported = false;
  return cudaSuccess;
}

template cudaError_t launch_stage_fused<float>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused<double>(const StageParams<double>&, int, int, cudaStream_t, bool*);

}  // namespace dh
