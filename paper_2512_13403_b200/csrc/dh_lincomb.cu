// dh_lincomb.cu — out = a X + b Y, elementwise over a state array.
//
// The stage kernels compute  out = B - tau D(U)  for ONE base state B.  The Shu-Osher forms of Heun's RK2 and
// SSPRK3 take convex combinations of two states as the base of their later stages
// (1/2 U + 1/2 U1;  3/4 U + 1/4 U1;  1/3 U + 2/3 U2), and their adjoints scale cotangents by the same weights;
// this streaming kernel forms those combinations (HBM-bound: 2 words read, 1 written per element; Y may be NULL
// for a pure scaling).  `out` may alias X or Y (each thread reads its elements before it writes them).
#include "dh_internal.cuh"

namespace dh {

template <class T> struct LVec;
template <> struct LVec<float> { using type = float4; static constexpr int W = 4; };
template <> struct LVec<double> { using type = double2; static constexpr int W = 2; };

template <class T>
__global__ void __launch_bounds__(256) lincomb_kernel(T* out, T a, const T* X, T b, const T* Y, size_t n) {
  using V = typename LVec<T>::type;
  constexpr int W = LVec<T>::W;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  const size_t nv = n / W;
  for (size_t v = tid; v < nv; v += nth) {
    V x = reinterpret_cast<const V*>(X)[v];
    T* px = reinterpret_cast<T*>(&x);
    if (Y) {
      V y = reinterpret_cast<const V*>(Y)[v];
      const T* py = reinterpret_cast<const T*>(&y);
#pragma unroll
      for (int l = 0; l < W; ++l) px[l] = a * px[l] + b * py[l];
    } else {
#pragma unroll
      for (int l = 0; l < W; ++l) px[l] = a * px[l];
    }
    reinterpret_cast<V*>(out)[v] = x;
  }
  for (size_t i = nv * W + tid; i < n; i += nth) out[i] = Y ? a * X[i] + b * Y[i] : a * X[i];
}

template <class T>
cudaError_t launch_lincomb(T* out, T a, const T* X, T b, const T* Y, size_t n, int sm_count, cudaStream_t s) {
  constexpr int W = LVec<T>::W;
  size_t want = (n / W + 255) / 256;
  const size_t cap = (size_t)sm_count * 8;
  int blocks = (int)(want < cap ? want : cap);
  if (blocks < 1) blocks = 1;
  lincomb_kernel<T><<<blocks, 256, 0, s>>>(out, a, X, b, Y, n);
  return cudaGetLastError();
}

template cudaError_t launch_lincomb<float>(float*, float, const float*, float, const float*, size_t, int, cudaStream_t);
template cudaError_t launch_lincomb<double>(double*, double, const double*, double, const double*, size_t, int, cudaStream_t);

}  // namespace dh
