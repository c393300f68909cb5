// dh_cfl.cu — CFL time step, Eq. A8: dt = C min_a dx_a / max_cells(|v_a| + c_s).
//
// Step a1 of SURVEY.md §8(a).  A grid-stride, vector-loading kernel evaluates the three wave speeds per
// cell with IEEE-rounded, never-contracted operations in T (the "dt recipe" of DESIGN.md), reduces them
// with warp shuffles and one shared-memory pass per block, and folds the block results into three global
// slots with atomicMax on the bit pattern (non-negative IEEE values order like unsigned integers, and
// max is exact and order independent, so the result is deterministic).  A one-thread epilogue kernel forms
// dt and re-arms the slots.  HBM-bound: 5 words read per cell, nothing written.
#include "dh_internal.cuh"

namespace dh {

// IEEE, non-contractable arithmetic in T
struct Ieee {
  static __device__ __forceinline__ float mul(float a, float b) { return __fmul_rn(a, b); }
  static __device__ __forceinline__ float add(float a, float b) { return __fadd_rn(a, b); }
  static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
  static __device__ __forceinline__ float div(float a, float b) { return __fdiv_rn(a, b); }
  static __device__ __forceinline__ float sqrt(float a) { return __fsqrt_rn(a); }
  static __device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
  static __device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
  static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
  static __device__ __forceinline__ double div(double a, double b) { return __ddiv_rn(a, b); }
  static __device__ __forceinline__ double sqrt(double a) { return __dsqrt_rn(a); }
};

__device__ __forceinline__ unsigned long long bits_of(float x) { return (unsigned long long)__float_as_uint(x); }
__device__ __forceinline__ unsigned long long bits_of(double x) { return (unsigned long long)__double_as_longlong(x); }
__device__ __forceinline__ void from_bits(unsigned long long b, float& x) { x = __uint_as_float((unsigned)b); }
__device__ __forceinline__ void from_bits(unsigned long long b, double& x) { x = __longlong_as_double((long long)b); }
__device__ __forceinline__ bool finite_(float x) { return isfinite(x); }
__device__ __forceinline__ bool finite_(double x) { return isfinite(x); }

template <class T>
__device__ __forceinline__ void cell_speeds(T rho, T mx, T my, T mz, T E, const CflParams<T>& p, T& sx, T& sy, T& sz, bool& bad) {
  const T rt = (rho >= p.rho_floor) ? rho : p.rho_floor;
  const T vx = Ieee::div(mx, rt), vy = Ieee::div(my, rt), vz = Ieee::div(mz, rt);
  const T q = Ieee::add(Ieee::add(Ieee::mul(mx, mx), Ieee::mul(my, my)), Ieee::mul(mz, mz));
  T P = Ieee::mul(p.gm1, Ieee::sub(E, Ieee::mul(T(0.5), Ieee::div(q, rt))));
  P = (P >= p.p_floor) ? P : p.p_floor;
  const T cs = Ieee::sqrt(Ieee::div(Ieee::mul(p.gamma, P), rt));
  const T ax = Ieee::add(abs_(vx), cs), ay = Ieee::add(abs_(vy), cs), az = Ieee::add(abs_(vz), cs);
  // the floors are compare-selects and would swallow a NaN in rho or E: test the inputs as well
  bad = bad || !(finite_(rho) && finite_(mx) && finite_(my) && finite_(mz) && finite_(E) && finite_(ax) && finite_(ay) && finite_(az));
  sx = (ax > sx) ? ax : sx;
  sy = (ay > sy) ? ay : sy;
  sz = (az > sz) ? az : sz;
}

template <class T> struct Vec;
template <> struct Vec<float> { using type = float4; static constexpr int W = 4; };
template <> struct Vec<double> { using type = double2; static constexpr int W = 2; };

template <class T>
__global__ void __launch_bounds__(256) cfl_reduce_kernel(const CflParams<T> p, const bool guarded) {
  using V = typename Vec<T>::type;
  constexpr int W = Vec<T>::W;
  const size_t N = p.N;
  if (guarded && p.cand_cnt[1] == 0u) return;      // the candidates already hold the maxima (cfl_cand_kernel)
  T sx = T(0), sy = T(0), sz = T(0);
  bool bad = false;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  if (N % W == 0) {
    const size_t nv = N / W;
    const V* r0 = reinterpret_cast<const V*>(p.U);
    const V* r1 = reinterpret_cast<const V*>(p.U + N);
    const V* r2 = reinterpret_cast<const V*>(p.U + 2 * N);
    const V* r3 = reinterpret_cast<const V*>(p.U + 3 * N);
    const V* r4 = reinterpret_cast<const V*>(p.U + 4 * N);
    for (size_t v = tid; v < nv; v += nth) {
      V a = __ldg(r0 + v), b = __ldg(r1 + v), c = __ldg(r2 + v), d = __ldg(r3 + v), e = __ldg(r4 + v);
      const T* pa = reinterpret_cast<const T*>(&a);
      const T* pb = reinterpret_cast<const T*>(&b);
      const T* pc = reinterpret_cast<const T*>(&c);
      const T* pd = reinterpret_cast<const T*>(&d);
      const T* pe = reinterpret_cast<const T*>(&e);
#pragma unroll
      for (int l = 0; l < W; ++l) cell_speeds<T>(pa[l], pb[l], pc[l], pd[l], pe[l], p, sx, sy, sz, bad);
    }
  } else {
    for (size_t i = tid; i < N; i += nth)
      cell_speeds<T>(p.U[i], p.U[N + i], p.U[2 * N + i], p.U[3 * N + i], p.U[4 * N + i], p, sx, sy, sz, bad);
  }
  // warp reduce (values are >= 0 or NaN; NaN handled through `bad`)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    T ox = __shfl_xor_sync(0xffffffffu, sx, o), oy = __shfl_xor_sync(0xffffffffu, sy, o), oz = __shfl_xor_sync(0xffffffffu, sz, o);
    sx = (ox > sx) ? ox : sx;
    sy = (oy > sy) ? oy : sy;
    sz = (oz > sz) ? oz : sz;
  }
  const unsigned anybad = __ballot_sync(0xffffffffu, bad);
  __shared__ T sm[3][8];
  __shared__ unsigned smbad[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { sm[0][warp] = sx; sm[1][warp] = sy; sm[2][warp] = sz; smbad[warp] = anybad; }
  __syncthreads();
  if (warp == 0) {
    const int nw = blockDim.x >> 5;
    sx = (lane < nw) ? sm[0][lane] : T(0);
    sy = (lane < nw) ? sm[1][lane] : T(0);
    sz = (lane < nw) ? sm[2][lane] : T(0);
    unsigned b = (lane < nw) ? smbad[lane] : 0u;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
      T ox = __shfl_xor_sync(0xffffffffu, sx, o), oy = __shfl_xor_sync(0xffffffffu, sy, o), oz = __shfl_xor_sync(0xffffffffu, sz, o);
      sx = (ox > sx) ? ox : sx;
      sy = (oy > sy) ? oy : sy;
      sz = (oz > sz) ? oz : sz;
      b |= __shfl_xor_sync(0xffffffffu, b, o);
    }
    if (lane == 0) {
      atomicMax(p.acc + 0, bits_of(sx));
      atomicMax(p.acc + 1, bits_of(sy));
      atomicMax(p.acc + 2, bits_of(sz));
      if (b) atomicOr(p.acc + 3, 1ull);
    }
  }
}

// Candidate path of dh_advance.  The last stage of the previous step appended every pack whose wave-speed ESTIMATE
// (fast math, from the values it was about to store) reached 0.999 theta, theta = 0.97 min_a S_a of the previous dt.
// This one-block kernel evaluates the exact dt recipe on those packs.  If the list did not overflow and the exact
// maximum of every axis reaches theta, no other cell can exceed it (their speeds are below theta) and the maxima
// are the global ones; otherwise the flag sends the guarded full reduction over the whole state.
template <class T>
__global__ void __launch_bounds__(1024) cfl_cand_kernel(const CflParams<T> p) {
  const unsigned cnt = p.cand_cnt[0];
  const unsigned n = cnt < p.cand_cap ? cnt : p.cand_cap;
  const size_t N = p.N;
  T sx = T(0), sy = T(0), sz = T(0);
  bool bad = false;
  for (unsigned i = threadIdx.x; i < n; i += blockDim.x) {
    const size_t cidx = p.cand_list[i];
#pragma unroll
    for (int l = 0; l < 2; ++l)
      cell_speeds<T>(p.U[cidx + l], p.U[N + cidx + l], p.U[2 * N + cidx + l], p.U[3 * N + cidx + l], p.U[4 * N + cidx + l], p, sx, sy, sz, bad);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    T ox = __shfl_xor_sync(0xffffffffu, sx, o), oy = __shfl_xor_sync(0xffffffffu, sy, o), oz = __shfl_xor_sync(0xffffffffu, sz, o);
    sx = (ox > sx) ? ox : sx;
    sy = (oy > sy) ? oy : sy;
    sz = (oz > sz) ? oz : sz;
  }
  const unsigned anybad = __ballot_sync(0xffffffffu, bad);
  __shared__ T sm[3][32];
  __shared__ unsigned smbad[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { sm[0][warp] = sx; sm[1][warp] = sy; sm[2][warp] = sz; smbad[warp] = anybad; }
  __syncthreads();
  if (warp == 0) {
    sx = sm[0][lane]; sy = sm[1][lane]; sz = sm[2][lane];
    unsigned b = smbad[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      T ox = __shfl_xor_sync(0xffffffffu, sx, o), oy = __shfl_xor_sync(0xffffffffu, sy, o), oz = __shfl_xor_sync(0xffffffffu, sz, o);
      sx = (ox > sx) ? ox : sx;
      sy = (oy > sy) ? oy : sy;
      sz = (oz > sz) ? oz : sz;
      b |= __shfl_xor_sync(0xffffffffu, b, o);
    }
    if (lane == 0) {
      atomicMax(p.acc + 0, bits_of(sx));
      atomicMax(p.acc + 1, bits_of(sy));
      atomicMax(p.acc + 2, bits_of(sz));
      if (b) atomicOr(p.acc + 3, 1ull);
      const T theta = p.cand_thr[1];
      const bool need = cnt > p.cand_cap || !(sx >= theta && sy >= theta && sz >= theta);
      p.cand_cnt[1] = need ? 1u : 0u;
      p.cand_stats[0] += 1ull;                 // one block, one thread: plain updates
      p.cand_stats[1] += need ? 1ull : 0ull;
      p.cand_stats[2] += n;
    }
  }
}

template <class T>
__global__ void cfl_finish_kernel(const CflParams<T> p) {
  T S[3];
  for (int a = 0; a < 3; ++a) { from_bits(p.acc[a], S[a]); p.acc[a] = 0ull; }
  const unsigned long long bad = p.acc[3];
  p.acc[3] = 0ull;
  T best = Ieee::div(p.dx[0], S[0]);
  for (int a = 1; a < 3; ++a) {
    const T r = Ieee::div(p.dx[a], S[a]);
    if (r < best) best = r;
  }
  const T dt = Ieee::mul(p.cfl, best);
  *p.dt_dev = dt;
  if (p.cand_thr) {          // thresholds for the candidates the next last stage will push, and an empty list
    T smin = S[0] < S[1] ? S[0] : S[1];
    smin = smin < S[2] ? smin : S[2];
    const T theta = T(0.97) * smin;
    p.cand_thr[1] = theta;
    p.cand_thr[0] = T(0.999) * theta;
    p.cand_cnt[0] = 0u;
    p.cand_cnt[1] = 0u;
  }
  p.result->smax[0] = (double)S[0];
  p.result->smax[1] = (double)S[1];
  p.result->smax[2] = (double)S[2];
  p.result->dt = (double)dt;
  p.result->nonfinite = bad;
}

template <class T>
cudaError_t launch_cfl_reduce(const CflParams<T>& p, int sm_count, cudaStream_t s) {
  constexpr int W = Vec<T>::W;
  size_t work = (p.N % W == 0) ? p.N / W : p.N;
  size_t want = (work + 255) / 256;
  size_t cap = (size_t)sm_count * 8;     // 8 resident 256-thread blocks per SM
  int blocks = (int)(want < cap ? want : cap);
  if (blocks < 1) blocks = 1;
  cfl_reduce_kernel<T><<<blocks, 256, 0, s>>>(p, false);
  return cudaGetLastError();
}

template <class T>
cudaError_t launch_cfl_candidates(const CflParams<T>& p, int sm_count, cudaStream_t s) {
  cfl_cand_kernel<T><<<1, 1024, 0, s>>>(p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  constexpr int W = Vec<T>::W;
  size_t work = (p.N % W == 0) ? p.N / W : p.N;
  size_t want = (work + 255) / 256;
  size_t cap = (size_t)sm_count * 8;
  int blocks = (int)(want < cap ? want : cap);
  if (blocks < 1) blocks = 1;
  cfl_reduce_kernel<T><<<blocks, 256, 0, s>>>(p, true);
  return cudaGetLastError();
}

template <class T>
cudaError_t launch_cfl_finish(const CflParams<T>& p, cudaStream_t s) {
  cfl_finish_kernel<T><<<1, 1, 0, s>>>(p);
  return cudaGetLastError();
}

template cudaError_t launch_cfl_reduce<float>(const CflParams<float>&, int, cudaStream_t);
template cudaError_t launch_cfl_reduce<double>(const CflParams<double>&, int, cudaStream_t);
template cudaError_t launch_cfl_candidates<float>(const CflParams<float>&, int, cudaStream_t);
template cudaError_t launch_cfl_candidates<double>(const CflParams<double>&, int, cudaStream_t);
template cudaError_t launch_cfl_finish<float>(const CflParams<float>&, cudaStream_t);
template cudaError_t launch_cfl_finish<double>(const CflParams<double>&, cudaStream_t);

}  // namespace dh
