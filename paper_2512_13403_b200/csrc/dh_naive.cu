// dh_naive.cu — one-thread-per-cell gather kernels (DH_OPT_KERNEL = 1).
//
// Same arithmetic as the fused z-sweep kernels, but every thread recomputes everything its cell needs
// straight from global memory with periodic index arithmetic: 13 primitive conversions, 9 slopes and 6 Riemann
// fluxes per cell-stage forward; 19 conversions, 15 slopes and 12 flux adjoints per cell-stage in reverse.
// Template parameters: the limiter (DH_OPT_LIMITER) and the Riemann flux (DH_OPT_RIEMANN: HLLC, HLL, Rusanov).
// They exist (a) as the in-library cross-check of the fused kernels, (b) as the path for grids the fused
// kernels do not cover, and (c) as the first correct reverse-mode path (gather form: no atomics,
// deterministic).  Steps a2-a7 of SURVEY.md §8(a).
#include "dh_internal.cuh"

namespace dh {

__device__ __forceinline__ int wrapi(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

template <class T>
__device__ __forceinline__ void load_prim(const T* __restrict__ U, size_t N, size_t cell, const Consts<T>& c, T W[5]) {
  T u[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) u[f] = U[f * N + cell];
  prim(u, c, W);
}

template <class T, int LIM>
__device__ __forceinline__ void slope(const T Wm[5], const T W0[5], const T Wp[5], T s[5]) {
#pragma unroll
  for (int q = 0; q < 5; ++q) s[q] = limit<T, LIM>(Wp[q] - W0[q], W0[q] - Wm[q]);
}

// acc -= coef * (F_{+1/2} - F_{-1/2}) along AX, from the five cells W[-2..2]
template <class T, int LIM, int RS, int AX>
__device__ __forceinline__ void axis_divergence(const T Wm2[5], const T Wm1[5], const T W0[5], const T Wp1[5],
                                                const T Wp2[5], const Consts<T>& c, T coef, T acc[5]) {
  T sm[5], s0[5], sp[5], L[5], R[5], Fm[5], Fp[5];
  slope<T, LIM>(Wm2, Wm1, W0, sm);
  slope<T, LIM>(Wm1, W0, Wp1, s0);
  slope<T, LIM>(W0, Wp1, Wp2, sp);
#pragma unroll
  for (int q = 0; q < 5; ++q) { L[q] = Wm1[q] + T(0.5) * sm[q]; R[q] = W0[q] - T(0.5) * s0[q]; }
  riemann_flux<T, AX, RS>(L, R, c, Fm);
#pragma unroll
  for (int q = 0; q < 5; ++q) { L[q] = W0[q] + T(0.5) * s0[q]; R[q] = Wp1[q] - T(0.5) * sp[q]; }
  riemann_flux<T, AX, RS>(L, R, c, Fp);
#pragma unroll
  for (int q = 0; q < 5; ++q) acc[q] -= coef * (Fp[q] - Fm[q]);
}

template <class T, int LIM, int RS>
__global__ void __launch_bounds__(128) stage_naive_kernel(const StageParams<T> p) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y, k = blockIdx.z;
  if (i >= p.nx) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const size_t N = (size_t)nx * ny * nz;
  const T dt = p.dt_dev ? *p.dt_dev : p.dt;
  const T tau = p.frac * dt;
  auto at = [&](int ii, int jj, int kk) { return ((size_t)kk * ny + jj) * nx + ii; };
  const size_t c0 = at(i, j, k);
  T W0[5], A[5], B[5], C[5], D[5], acc[5];
  load_prim(p.U, N, c0, p.c, W0);
#pragma unroll
  for (int f = 0; f < 5; ++f) acc[f] = p.B[f * N + c0];
  load_prim(p.U, N, at(wrapi(i - 2, nx), j, k), p.c, A);
  load_prim(p.U, N, at(wrapi(i - 1, nx), j, k), p.c, B);
  load_prim(p.U, N, at(wrapi(i + 1, nx), j, k), p.c, C);
  load_prim(p.U, N, at(wrapi(i + 2, nx), j, k), p.c, D);
  axis_divergence<T, LIM, RS, 0>(A, B, W0, C, D, p.c, tau * p.inv_dx[0], acc);
  load_prim(p.U, N, at(i, wrapi(j - 2, ny), k), p.c, A);
  load_prim(p.U, N, at(i, wrapi(j - 1, ny), k), p.c, B);
  load_prim(p.U, N, at(i, wrapi(j + 1, ny), k), p.c, C);
  load_prim(p.U, N, at(i, wrapi(j + 2, ny), k), p.c, D);
  axis_divergence<T, LIM, RS, 1>(A, B, W0, C, D, p.c, tau * p.inv_dx[1], acc);
  load_prim(p.U, N, at(i, j, wrapi(k - 2, nz)), p.c, A);
  load_prim(p.U, N, at(i, j, wrapi(k - 1, nz)), p.c, B);
  load_prim(p.U, N, at(i, j, wrapi(k + 1, nz)), p.c, C);
  load_prim(p.U, N, at(i, j, wrapi(k + 2, nz)), p.c, D);
  axis_divergence<T, LIM, RS, 2>(A, B, W0, C, D, p.c, tau * p.inv_dx[2], acc);
  if (p.cool) acc[4] = cool_energy(acc, dt, p.c);
#pragma unroll
  for (int f = 0; f < 5; ++f) p.out[f * N + c0] = acc[f];
}

// Wb += contribution of axis AX to the cotangent of W at the centre cell.
// W[0..6] = cells i-3..i+3 along the axis, g[0..4] = cotangent at cells i-2..i+2, coef = tau/dx.
template <class T, int LIM, int RS, int AX>
__device__ __forceinline__ void axis_vjp(const T (&W)[7][5], const T (&g)[5][5], const Consts<T>& c, T coef, T Wb[5]) {
  T s[5][5];          // slopes of cells i-2..i+2
#pragma unroll
  for (int m = 0; m < 5; ++m) slope<T, LIM>(W[m], W[m + 1], W[m + 2], s[m]);
  T WLb[4][5], WRb[4][5];   // face j lies between cells (i-2+j, i-1+j)
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    T L[5], R[5], lam[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      L[q] = W[j + 1][q] + T(0.5) * s[j][q];
      R[q] = W[j + 2][q] - T(0.5) * s[j + 1][q];
      lam[q] = coef * (g[j + 1][q] - g[j][q]);
      WLb[j][q] = T(0);
      WRb[j][q] = T(0);
    }
    riemann_flux_vjp<T, AX, RS>(L, R, c, lam, WLb[j], WRb[j]);
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    // slope cotangents of cells i-1, i, i+1  (cell m=i-2+.. has right face j=m, left face j=m-1 in 0-based cell index)
    const T Sbm = T(0.5) * (WLb[1][q] - WRb[0][q]);   // cell i-1: right face j=1, left face j=0
    const T Sb0 = T(0.5) * (WLb[2][q] - WRb[1][q]);   // cell i
    const T Sbp = T(0.5) * (WLb[3][q] - WRb[2][q]);   // cell i+1
    T dam, dbm, da0, db0, dap, dbp;
    limit_grad<T, LIM>(W[3][q] - W[2][q], W[2][q] - W[1][q], dam, dbm);   // cell i-1: a = W_i - W_{i-1}
    limit_grad<T, LIM>(W[4][q] - W[3][q], W[3][q] - W[2][q], da0, db0);   // cell i
    limit_grad<T, LIM>(W[5][q] - W[4][q], W[4][q] - W[3][q], dap, dbp);   // cell i+1: b = W_{i+1} - W_i
    (void)dbm; (void)dap;
    Wb[q] += WLb[2][q] + WRb[1][q] + dam * Sbm + (db0 - da0) * Sb0 - dbp * Sbp;
  }
}

template <class T, int LIM, int RS>
__global__ void __launch_bounds__(64) rev_naive_kernel(const RevParams<T> p) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y, k = blockIdx.z;
  if (i >= p.nx) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const size_t N = (size_t)nx * ny * nz;
  const T tau = p.frac * p.dt;
  auto at = [&](int ii, int jj, int kk) { return ((size_t)kk * ny + jj) * nx + ii; };
  const size_t c0 = at(i, j, k);
  T W[7][5], g[5][5], Wb[5] = {T(0), T(0), T(0), T(0), T(0)};
  T Wc[5], gc[5];
  load_prim(p.U, N, c0, p.c, Wc);
#pragma unroll
  for (int f = 0; f < 5; ++f) gc[f] = p.g[f * N + c0];

#pragma unroll
  for (int m = 0; m < 7; ++m) {
    if (m == 3) { for (int f = 0; f < 5; ++f) W[3][f] = Wc[f]; }
    else load_prim(p.U, N, at(wrapi(wrapi(i + m - 3, nx), nx), j, k), p.c, W[m]);
  }
#pragma unroll
  for (int m = 0; m < 5; ++m)
    for (int f = 0; f < 5; ++f) g[m][f] = (m == 2) ? gc[f] : p.g[f * N + at(wrapi(i + m - 2, nx), j, k)];
  axis_vjp<T, LIM, RS, 0>(W, g, p.c, tau * p.inv_dx[0], Wb);

#pragma unroll
  for (int m = 0; m < 7; ++m)
    if (m != 3) load_prim(p.U, N, at(i, wrapi(wrapi(j + m - 3, ny), ny), k), p.c, W[m]);
#pragma unroll
  for (int m = 0; m < 5; ++m)
    for (int f = 0; f < 5; ++f) g[m][f] = (m == 2) ? gc[f] : p.g[f * N + at(i, wrapi(j + m - 2, ny), k)];
  axis_vjp<T, LIM, RS, 1>(W, g, p.c, tau * p.inv_dx[1], Wb);

#pragma unroll
  for (int m = 0; m < 7; ++m)
    if (m != 3) load_prim(p.U, N, at(i, j, wrapi(wrapi(k + m - 3, nz), nz)), p.c, W[m]);
#pragma unroll
  for (int m = 0; m < 5; ++m)
    for (int f = 0; f < 5; ++f) g[m][f] = (m == 2) ? gc[f] : p.g[f * N + at(i, j, wrapi(k + m - 2, nz))];
  axis_vjp<T, LIM, RS, 2>(W, g, p.c, tau * p.inv_dx[2], Wb);

  T u[5], Ub[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) u[f] = p.U[f * N + c0];
  prim_vjp(u, p.c, Wb, Ub);
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    T v = Ub[f];
    if (p.b1) v += p.w1 * p.b1[f * N + c0];
    if (p.b2) v += p.w2 * p.b2[f * N + c0];
    p.out[f * N + c0] = v;
  }
}

constexpr int DH_TAB_MAX = 256;

// the table of the two-branch law into shared memory (DH_OPT_COOL_LAW = 1); returns the Consts to use in this block
template <class T>
__device__ __forceinline__ Consts<T> stage_table(const Consts<T>& c, T* stab) {
  Consts<T> cc = c;
  if (c.cool_law != 0) {
    for (int i = threadIdx.x; i < c.ntab; i += blockDim.x) stab[i] = c.tab[i];
    __syncthreads();
    cc.tab = stab;
  }
  return cc;
}

template <class T>
__global__ void __launch_bounds__(256) cool_vjp_kernel(const T* __restrict__ U1, const T* __restrict__ g, T* __restrict__ gout,
                                                       size_t N, T dt, Consts<T> c) {
  __shared__ T stab[DH_TAB_MAX];
  const Consts<T> cc = stage_table(c, stab);
  const bool general = cc.cool_mode != 0 || cc.cool_nsub > 1 || cc.cool_law != 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
    T u[5], gi[5], gb[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) { u[f] = U1[f * N + i]; gi[f] = g[f * N + i]; }
    if (general) cool_vjp_general(u, dt, cc, gi, gb); else cool_vjp(u, dt, cc, gi, gb);
#pragma unroll
    for (int f = 0; f < 5; ++f) gout[f * N + i] = gb[f];
  }
}

// Gradient of sum(g_E * E_out) with respect to the table nodes, at the pre-cooling state U1: every block
// accumulates the contributions of its cells in shared memory (fp64), writes its partial sums, and cool_table_sum_kernel
// adds the blocks in a fixed order.
template <class T>
__global__ void __launch_bounds__(256) cool_table_vjp_kernel(const T* __restrict__ U1, const T* __restrict__ g, size_t N, T dt, Consts<T> c,
                                                             double* __restrict__ part) {
  __shared__ T stab[DH_TAB_MAX];
  __shared__ double acc[DH_TAB_MAX];
  for (int i = threadIdx.x; i < c.ntab; i += blockDim.x) acc[i] = 0.0;
  const Consts<T> cc = stage_table(c, stab);          // (its barrier also publishes the zeroed accumulator)
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
    T u[5], gi[5], gb[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) { u[f] = U1[f * N + i]; gi[f] = (f == 4) ? g[f * N + i] : T(0); }
    cool_vjp_general(u, dt, cc, gi, gb, acc);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < c.ntab; i += blockDim.x) part[(size_t)blockIdx.x * c.ntab + i] = acc[i];
}

__global__ void cool_table_sum_kernel(const double* __restrict__ part, int nblocks, int ntab, double scale, double* __restrict__ out) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= ntab) return;
  double s = 0.0;
  for (int b = 0; b < nblocks; ++b) s += part[(size_t)b * ntab + k];
  out[k] = s * scale;
}

// limiter in {0, 1, 2} x riemann in {0, 1, 2} -> one instantiation each
#define DH_NAIVE_DISPATCH(KERNEL, ...)                                        \
  switch (limiter * 3 + riemann) {                                            \
    case 1: KERNEL<T, 0, 1><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 2: KERNEL<T, 0, 2><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 3: KERNEL<T, 1, 0><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 4: KERNEL<T, 1, 1><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 5: KERNEL<T, 1, 2><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 6: KERNEL<T, 2, 0><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 7: KERNEL<T, 2, 1><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    case 8: KERNEL<T, 2, 2><<<grid, block, 0, s>>>(__VA_ARGS__); break;       \
    default: KERNEL<T, 0, 0><<<grid, block, 0, s>>>(__VA_ARGS__); break;      \
  }

template <class T>
cudaError_t launch_stage_naive(const StageParams<T>& p, int limiter, int riemann, cudaStream_t s) {
  dim3 block(128), grid((p.nx + 127) / 128, p.ny, p.nz);
  DH_NAIVE_DISPATCH(stage_naive_kernel, p)
  return cudaGetLastError();
}

template <class T>
cudaError_t launch_rev_naive(const RevParams<T>& p, int limiter, int riemann, cudaStream_t s) {
  dim3 block(64), grid((p.nx + 63) / 64, p.ny, p.nz);
  DH_NAIVE_DISPATCH(rev_naive_kernel, p)
  return cudaGetLastError();
}

// In-place cooling of a finished state for the integrators the stage kernels do not fuse (sub-cycled Eq. 23, trapezoid
// Eq. 22; DH_OPT_COOL_MODE / DH_OPT_COOL_NSUB): reads the 5 fields, rewrites E.  dt from the device when dt_dev != NULL.
template <class T>
__global__ void __launch_bounds__(256) cool_fwd_kernel(T* __restrict__ U, size_t N, T dt_host, const T* __restrict__ dt_dev, Consts<T> c) {
  __shared__ T stab[DH_TAB_MAX];
  const Consts<T> cc = stage_table(c, stab);
  const T dt = dt_dev ? *dt_dev : dt_host;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
    T u[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) u[f] = U[f * N + i];
    U[4 * N + i] = cool_energy_general(u, dt, cc);
  }
}

template <class T>
cudaError_t launch_cool_fwd(T* U, size_t N, T dt, const T* dt_dev, const Consts<T>& c, cudaStream_t s) {
  int blocks = (int)((N + 255) / 256);
  if (blocks > 148 * 16) blocks = 148 * 16;
  cool_fwd_kernel<T><<<blocks, 256, 0, s>>>(U, N, dt, dt_dev, c);
  return cudaGetLastError();
}

template <class T>
cudaError_t launch_cool_vjp(const T* U1, const T* g, T* gout, size_t N, T dt, const Consts<T>& c, cudaStream_t s) {
  int blocks = (int)((N + 255) / 256);
  if (blocks > 148 * 16) blocks = 148 * 16;
  cool_vjp_kernel<T><<<blocks, 256, 0, s>>>(U1, g, gout, N, dt, c);
  return cudaGetLastError();
}

// gtab (DEVICE, ntab doubles) = d sum(g_E E_out) / d (log10 Lambda at the nodes); part: DEVICE scratch of cool_table_blocks() x ntab
int cool_table_blocks() { return 148 * 4; }

template <class T>
cudaError_t launch_cool_table_vjp(const T* U1, const T* g, size_t N, T dt, const Consts<T>& c, double* part, double* gtab, cudaStream_t s) {
  int blocks = (int)((N + 255) / 256);
  if (blocks > cool_table_blocks()) blocks = cool_table_blocks();
  cool_table_vjp_kernel<T><<<blocks, 256, 0, s>>>(U1, g, N, dt, c, part);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  // the table is held as log2 Lambda: d / d log10 Lambda = log2(10) d / d log2 Lambda
  cool_table_sum_kernel<<<(c.ntab + 63) / 64, 64, 0, s>>>(part, blocks, c.ntab, 3.321928094887362, gtab);
  return cudaGetLastError();
}

template cudaError_t launch_cool_table_vjp<float>(const float*, const float*, size_t, float, const Consts<float>&, double*, double*, cudaStream_t);
template cudaError_t launch_cool_table_vjp<double>(const double*, const double*, size_t, double, const Consts<double>&, double*, double*, cudaStream_t);
template cudaError_t launch_stage_naive<float>(const StageParams<float>&, int, int, cudaStream_t);
template cudaError_t launch_stage_naive<double>(const StageParams<double>&, int, int, cudaStream_t);
template cudaError_t launch_rev_naive<float>(const RevParams<float>&, int, int, cudaStream_t);
template cudaError_t launch_rev_naive<double>(const RevParams<double>&, int, int, cudaStream_t);
template cudaError_t launch_cool_fwd<float>(float*, size_t, float, const float*, const Consts<float>&, cudaStream_t);
template cudaError_t launch_cool_fwd<double>(double*, size_t, double, const double*, const Consts<double>&, cudaStream_t);
template cudaError_t launch_cool_vjp<float>(const float*, const float*, float*, size_t, float, const Consts<float>&, cudaStream_t);
template cudaError_t launch_cool_vjp<double>(const double*, const double*, double*, size_t, double, const Consts<double>&, cudaStream_t);

}  // namespace dh
