// dh_gravity.cu — self-gravity as a source term of the hydro step (§6; the force-class form of
// PAPER.md:88-107): with the potential phi of Eq. 27 (from the multigrid solver of dh_poisson.cu),
//     g_a = -(phi_{i+1} - phi_{i-1}) / (2 dx_a)            "the usual finite-difference gradient" (reading A27)
//     u <- u + s_g dt,   s_g = (0, rho g, m . g)            momentum and energy sources, from the incoming u
// and the transposes of both maps.  Streaming kernels, one thread per cell; phi is read through L1 / L2 (7-point pattern).
// Algorithmic words per cell: source 5 read + 4 written + 1 (phi) = 10; VJP 5 (U) + 5 (g_out) + 1 (phi) in, 5 + 1 out.
#include "dh_internal.cuh"

namespace dh {

namespace {

struct Nbr { size_t xm, xp, ym, yp, zm, zp; };
__device__ __forceinline__ Nbr neighbours(size_t c, int nx, int ny, int nz) {
  const size_t NP = (size_t)nx * ny;
  const int k = (int)(c / NP);
  const size_t rem = c - (size_t)k * NP;
  const int j = (int)(rem / nx), i = (int)(rem - (size_t)j * nx);
  Nbr n;
  n.xm = c - i + (i == 0 ? nx - 1 : i - 1);
  n.xp = c - i + (i == nx - 1 ? 0 : i + 1);
  n.ym = c - (size_t)j * nx + (size_t)(j == 0 ? ny - 1 : j - 1) * nx;
  n.yp = c - (size_t)j * nx + (size_t)(j == ny - 1 ? 0 : j + 1) * nx;
  n.zm = c - (size_t)k * NP + (size_t)(k == 0 ? nz - 1 : k - 1) * NP;
  n.zp = c - (size_t)k * NP + (size_t)(k == nz - 1 ? 0 : k + 1) * NP;
  return n;
}

template <class T>
__global__ void __launch_bounds__(256) grav_rhs_kernel(const T* __restrict__ rho, T* __restrict__ F, size_t N, T four_pi_g) {
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) F[c] = four_pi_g * rho[c];
}

// grho[c] += 4 pi G gF[c]:  transpose of F = 4 pi G rho.  (The solver works on the zero-mean part of F, reading A23; the transpose
// of that projection is applied by the adjoint solve itself, which returns a zero-mean gF.)
template <class T>
__global__ void __launch_bounds__(256) grav_rhs_vjp_kernel(const T* __restrict__ gF, T* __restrict__ grho, size_t N, T four_pi_g) {
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) grho[c] += four_pi_g * gF[c];
}

template <class T>
__global__ void __launch_bounds__(256) grav_source_kernel(T* __restrict__ U, const T* __restrict__ phi, int nx, int ny, int nz, T hx, T hy, T hz,
                                                          T dt_host, const T* __restrict__ dt_dev) {
  const size_t N = (size_t)nx * ny * nz;
  const T dt = dt_dev ? *dt_dev : dt_host;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
    const Nbr n = neighbours(c, nx, ny, nz);
    const T gx = -(phi[n.xp] - phi[n.xm]) * hx, gy = -(phi[n.yp] - phi[n.ym]) * hy, gz = -(phi[n.zp] - phi[n.zm]) * hz;   // h_a = 1 / (2 dx_a)
    const T rho = U[c], mx = U[N + c], my = U[2 * N + c], mz = U[3 * N + c];
    U[N + c] = mx + dt * rho * gx;
    U[2 * N + c] = my + dt * rho * gy;
    U[3 * N + c] = mz + dt * rho * gz;
    U[4 * N + c] += dt * (mx * gx + my * gy + mz * gz);
  }
}

// pass 1 of the transpose: dL/dU (needs g at the cell) and the cotangents of the three acceleration components
// gb_a = dt (rho gout_{m_a} + m_a gout_E), kept in `gb` [3][N]; pass 2 turns them into dL/dphi by the transposed differences
template <class T>
__global__ void __launch_bounds__(256) grav_source_vjp_kernel(const T* __restrict__ U, const T* __restrict__ phi, const T* __restrict__ gout,
                                                              T* __restrict__ gin, T* __restrict__ gb, int nx, int ny, int nz, T hx, T hy, T hz, T dt) {
  const size_t N = (size_t)nx * ny * nz;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
    const Nbr n = neighbours(c, nx, ny, nz);
    const T gx = -(phi[n.xp] - phi[n.xm]) * hx, gy = -(phi[n.yp] - phi[n.ym]) * hy, gz = -(phi[n.zp] - phi[n.zm]) * hz;
    const T rho = U[c], mx = U[N + c], my = U[2 * N + c], mz = U[3 * N + c];
    const T o0 = gout[c], o1 = gout[N + c], o2 = gout[2 * N + c], o3 = gout[3 * N + c], o4 = gout[4 * N + c];
    gin[c] = o0 + dt * (gx * o1 + gy * o2 + gz * o3);
    gin[N + c] = o1 + dt * gx * o4;
    gin[2 * N + c] = o2 + dt * gy * o4;
    gin[3 * N + c] = o3 + dt * gz * o4;
    gin[4 * N + c] = o4;
    gb[c] = dt * (rho * o1 + mx * o4);
    gb[N + c] = dt * (rho * o2 + my * o4);
    gb[2 * N + c] = dt * (rho * o3 + mz * o4);
  }
}

template <class T>
__global__ void __launch_bounds__(256) grav_phi_vjp_kernel(const T* __restrict__ gb, T* __restrict__ gphi, int nx, int ny, int nz, T hx, T hy, T hz) {
  const size_t N = (size_t)nx * ny * nz;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < N; c += (size_t)gridDim.x * blockDim.x) {
    const Nbr n = neighbours(c, nx, ny, nz);
    gphi[c] = (gb[n.xp] - gb[n.xm]) * hx + (gb[N + n.yp] - gb[N + n.ym]) * hy + (gb[2 * N + n.zp] - gb[2 * N + n.zm]) * hz;
  }
}

int grid_for(size_t N) {
  size_t b = (N + 255) / 256;
  return (int)(b > 148 * 16 ? 148 * 16 : b);
}

}  // namespace

template <class T>
cudaError_t launch_grav_rhs(const T* rho, T* F, size_t N, T four_pi_g, cudaStream_t s) {
  grav_rhs_kernel<T><<<grid_for(N), 256, 0, s>>>(rho, F, N, four_pi_g);
  return cudaGetLastError();
}
template <class T>
cudaError_t launch_grav_rhs_vjp(const T* gF, T* grho, size_t N, T four_pi_g, cudaStream_t s) {
  grav_rhs_vjp_kernel<T><<<grid_for(N), 256, 0, s>>>(gF, grho, N, four_pi_g);
  return cudaGetLastError();
}
template <class T>
cudaError_t launch_grav_source(T* U, const T* phi, int nx, int ny, int nz, const double dx[3], T dt, const T* dt_dev, cudaStream_t s) {
  grav_source_kernel<T><<<grid_for((size_t)nx * ny * nz), 256, 0, s>>>(U, phi, nx, ny, nz, (T)(0.5 / dx[0]), (T)(0.5 / dx[1]), (T)(0.5 / dx[2]), dt, dt_dev);
  return cudaGetLastError();
}
template <class T>
cudaError_t launch_grav_source_vjp(const T* U, const T* phi, const T* gout, T* gin, T* gb, T* gphi, int nx, int ny, int nz, const double dx[3], T dt, cudaStream_t s) {
  const T hx = (T)(0.5 / dx[0]), hy = (T)(0.5 / dx[1]), hz = (T)(0.5 / dx[2]);
  const int g = grid_for((size_t)nx * ny * nz);
  grav_source_vjp_kernel<T><<<g, 256, 0, s>>>(U, phi, gout, gin, gb, nx, ny, nz, hx, hy, hz, dt);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  grav_phi_vjp_kernel<T><<<g, 256, 0, s>>>(gb, gphi, nx, ny, nz, hx, hy, hz);
  return cudaGetLastError();
}

#define DH_INST(T)                                                                                                     \
  template cudaError_t launch_grav_rhs<T>(const T*, T*, size_t, T, cudaStream_t);                                      \
  template cudaError_t launch_grav_rhs_vjp<T>(const T*, T*, size_t, T, cudaStream_t);                                  \
  template cudaError_t launch_grav_source<T>(T*, const T*, int, int, int, const double*, T, const T*, cudaStream_t);   \
  template cudaError_t launch_grav_source_vjp<T>(const T*, const T*, const T*, T*, T*, T*, int, int, int, const double*, T, cudaStream_t);
DH_INST(float)
DH_INST(double)
#undef DH_INST

}  // namespace dh
