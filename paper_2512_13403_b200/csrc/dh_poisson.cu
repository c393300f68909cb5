// dh_poisson.cu — periodic geometric multigrid for the seven-point Poisson problem A phi = F (sm_100a).
//
// PAPER.md §6.2 (Eqs. 37-48) and Appendix C: weighted Jacobi smoothing (Eq. 39, omega = 2/3), residual (Eq. 41),
// cell-centred full-weighting restriction (Eq. 42), trilinear prolongation + correction (Eqs. 44-45), V / W cycles
// (Eqs. C10-C12), and the adjoint as another solve (Eqs. 46-48).  Readings A21-A23 of DESIGN.md: Eq. 39 wins over the
// misprinted Eq. 40; the coarsest level (first level with an odd or 2-cell extent: 2^3 for power-of-two grids) is "solved" by nu_coarse Jacobi
// sweeps from zero; the solve works on the zero-mean part of F and returns the zero-mean phi.
//
// Every operator is an HBM-bound stencil: no tensor cores.  Kernels:
//   mg_jacobi_kernel            out = (1-w) in + (w/6) (sum of 6 neighbours - h^2 F); 4 x-adjacent cells per thread,
//                               16-byte loads / stores (algorithmic 3 words per cell: in, F, out)
//   mg_residual_restrict_kernel r2h = mean over the 8 children of (F - A phi): residual and restriction fused, the fine
//                               residual never reaches HBM (algorithmic 2 words per fine cell + 1/8 written)
//   mg_prolong_add_kernel       phi += P e2h: one thread per coarse cell writes its 2x2x2 children (27 coarse reads from
//                               L1 / L2; algorithmic 2 words per fine cell + 1/8 read)
//   mg_subtree_kernel           a level of <= 4096 cells and all levels below it in ONE block (DH_MG_SUBTREE, default)
//   mg_coarse_kernel            the coarsest level in ONE block: nu_coarse sweeps in shared memory (<= 1024 cells)
//   mg_sum_kernel / mg_sum_finish_kernel / mg_shift_kernel   deterministic mean (fixed-order two-stage sum in fp64)
//   mg_resnorm_kernel           |F - A phi|^2 and |F|^2 for the reported relative residual (two-stage, deterministic)
// A cycle is captured once into a CUDA graph per (phi, F) pointer pair: the coarse levels are launch bound (a W-cycle
// at 512^3 is 1786 launches one per operator, 218 with the coarse levels in one block: mg_subtree_kernel).
#include <cstdio>
#include <vector>

#include "../../include/dh.h"
#include "dh_internal.cuh"

namespace dh {
void set_error(const char* where, const char* detail);   // dh_api.cu: the text dh_last_error() returns
}

namespace {

using dh::set_error;

__device__ __forceinline__ int wrp(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

template <class T> struct V4 { T a, b, c, d; };
template <> struct alignas(16) V4<float> { float a, b, c, d; };
template <> struct alignas(32) V4<double> { double a, b, c, d; };

// ---------------------------------------------------------------------------------------------- Jacobi (Eq. 39)
// VEC = 4: nx % 4 == 0, one thread per 4 cells; VEC = 1: any nx.  zero_in: `in` is identically zero (first sweep of an
// error equation) and is not read.
template <class T, int VEC>
__global__ void __launch_bounds__(128) mg_jacobi_kernel(T* __restrict__ out, const T* __restrict__ in, const T* __restrict__ F,
                                                        int nx, int ny, int nz, T c0, T c1, T h2, int zero_in) {
  const int i0 = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;
  const int j = blockIdx.y, k = blockIdx.z;
  if (i0 >= nx) return;
  const size_t row = ((size_t)k * ny + j) * nx;
  if (VEC == 4) {
    const V4<T> f = *reinterpret_cast<const V4<T>*>(F + row + i0);
    V4<T> o;
    if (zero_in) {
      o.a = -c1 * h2 * f.a; o.b = -c1 * h2 * f.b; o.c = -c1 * h2 * f.c; o.d = -c1 * h2 * f.d;
    } else {
      const size_t rym = ((size_t)k * ny + wrp(j - 1, ny)) * nx, ryp = ((size_t)k * ny + wrp(j + 1, ny)) * nx;
      const size_t rzm = ((size_t)wrp(k - 1, nz) * ny + j) * nx, rzp = ((size_t)wrp(k + 1, nz) * ny + j) * nx;
      const V4<T> c = *reinterpret_cast<const V4<T>*>(in + row + i0);
      const V4<T> ym = *reinterpret_cast<const V4<T>*>(in + rym + i0), yp = *reinterpret_cast<const V4<T>*>(in + ryp + i0);
      const V4<T> zm = *reinterpret_cast<const V4<T>*>(in + rzm + i0), zp = *reinterpret_cast<const V4<T>*>(in + rzp + i0);
      const T xl = in[row + wrp(i0 - 1, nx)], xr = in[row + wrp(i0 + 4, nx)];
      o.a = c0 * c.a + c1 * ((((xl + c.b) + (ym.a + yp.a)) + (zm.a + zp.a)) - h2 * f.a);
      o.b = c0 * c.b + c1 * ((((c.a + c.c) + (ym.b + yp.b)) + (zm.b + zp.b)) - h2 * f.b);
      o.c = c0 * c.c + c1 * ((((c.b + c.d) + (ym.c + yp.c)) + (zm.c + zp.c)) - h2 * f.c);
      o.d = c0 * c.d + c1 * ((((c.c + xr) + (ym.d + yp.d)) + (zm.d + zp.d)) - h2 * f.d);
    }
    *reinterpret_cast<V4<T>*>(out + row + i0) = o;
  } else {
    const T f = F[row + i0];
    T o;
    if (zero_in) {
      o = -c1 * h2 * f;
    } else {
      const T s = ((in[row + wrp(i0 - 1, nx)] + in[row + wrp(i0 + 1, nx)]) +
                   (in[((size_t)k * ny + wrp(j - 1, ny)) * nx + i0] + in[((size_t)k * ny + wrp(j + 1, ny)) * nx + i0])) +
                  (in[((size_t)wrp(k - 1, nz) * ny + j) * nx + i0] + in[((size_t)wrp(k + 1, nz) * ny + j) * nx + i0]);
      o = c0 * in[row + i0] + c1 * (s - h2 * f);
    }
    out[row + i0] = o;
  }
}

// --------------------------------------------------------------- residual (Eq. 41) + restriction (Eq. 42), fused
// one thread per coarse cell (I, J, K): r2h = 1/8 sum over the 8 children of F - (nbr sum - 6 phi) / h^2
template <class T>
__global__ void __launch_bounds__(128) mg_residual_restrict_kernel(T* __restrict__ rc, const T* __restrict__ phi, const T* __restrict__ F,
                                                                   int nx, int ny, int nz, T inv_h2) {
  const int I = blockIdx.x * blockDim.x + threadIdx.x;
  const int J = blockIdx.y, K = blockIdx.z;
  const int cx = nx >> 1, cy = ny >> 1;
  if (I >= cx) return;
  const int i = 2 * I, im = wrp(i - 1, nx), ip = wrp(i + 2, nx);
  T acc = T(0);
#pragma unroll
  for (int dk = 0; dk < 2; ++dk) {
#pragma unroll
    for (int dj = 0; dj < 2; ++dj) {
      const int j = 2 * J + dj, k = 2 * K + dk;
      const size_t row = ((size_t)k * ny + j) * nx;
      const size_t rym = ((size_t)k * ny + wrp(j - 1, ny)) * nx, ryp = ((size_t)k * ny + wrp(j + 1, ny)) * nx;
      const size_t rzm = ((size_t)wrp(k - 1, nz) * ny + j) * nx, rzp = ((size_t)wrp(k + 1, nz) * ny + j) * nx;
      const T c0 = phi[row + i], c1 = phi[row + i + 1];
      const T s0 = ((phi[row + im] + c1) + (phi[rym + i] + phi[ryp + i])) + (phi[rzm + i] + phi[rzp + i]);
      const T s1 = ((c0 + phi[row + ip]) + (phi[rym + i + 1] + phi[ryp + i + 1])) + (phi[rzm + i + 1] + phi[rzp + i + 1]);
      acc += (F[row + i] - (s0 - T(6) * c0) * inv_h2) + (F[row + i + 1] - (s1 - T(6) * c1) * inv_h2);
    }
  }
  rc[((size_t)K * cy + J) * cx + I] = T(0.125) * acc;
}

// --------------------------------------------------- prolongation (Eq. 44) + correction (Eq. 45): phi += P e
// one thread per coarse cell: its 2x2x2 children; per axis child 0 takes 3/4 e[I] + 1/4 e[I-1], child 1 3/4 e[I] + 1/4 e[I+1]
template <class T>
__global__ void __launch_bounds__(128) mg_prolong_add_kernel(T* __restrict__ phi, const T* __restrict__ e, int nx, int ny, int nz) {
  const int I = blockIdx.x * blockDim.x + threadIdx.x;
  const int J = blockIdx.y, K = blockIdx.z;
  const int cx = nx >> 1, cy = ny >> 1, cz = nz >> 1;
  if (I >= cx) return;
  const int Is[3] = {wrp(I - 1, cx), I, wrp(I + 1, cx)};
  const int Js[3] = {wrp(J - 1, cy), J, wrp(J + 1, cy)};
  const int Ks[3] = {wrp(K - 1, cz), K, wrp(K + 1, cz)};
  // interpolate along x first: for every (dz, dy) of the 3x3 coarse rows, the two x children
  T x0[3][3], x1[3][3];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      const T* r = e + ((size_t)Ks[a] * cy + Js[b]) * cx;
      const T m = r[Is[0]], c = r[Is[1]], p = r[Is[2]];
      x0[a][b] = T(0.75) * c + T(0.25) * m;
      x1[a][b] = T(0.75) * c + T(0.25) * p;
    }
#pragma unroll
  for (int dk = 0; dk < 2; ++dk)
#pragma unroll
    for (int dj = 0; dj < 2; ++dj) {
      const int kn = dk ? 2 : 0, jn = dj ? 2 : 0;     // the neighbour row each child leans towards
      const T y0c = T(0.75) * x0[1][1] + T(0.25) * x0[1][jn], y0n = T(0.75) * x0[kn][1] + T(0.25) * x0[kn][jn];
      const T y1c = T(0.75) * x1[1][1] + T(0.25) * x1[1][jn], y1n = T(0.75) * x1[kn][1] + T(0.25) * x1[kn][jn];
      const size_t o = ((size_t)(2 * K + dk) * ny + (2 * J + dj)) * nx + 2 * I;
      phi[o] += T(0.75) * y0c + T(0.25) * y0n;
      phi[o + 1] += T(0.75) * y1c + T(0.25) * y1n;
    }
}

// ------------------------------------------- coarsest level: nu sweeps (from zero, or from `init`) in one block
template <class T>
__global__ void __launch_bounds__(1024) mg_coarse_kernel(T* out, const T* init, const T* __restrict__ F, int nx, int ny, int nz,
                                                         T c0, T c1, T h2, int nu) {
  __shared__ T buf[2][1024];
  const int n = nx * ny * nz, t = threadIdx.x;
  const int i = t % nx, j = (t / nx) % ny, k = t / (nx * ny);
  const bool on = t < n;
  const T f = on ? F[t] : T(0);
  int nb[6] = {0, 0, 0, 0, 0, 0};
  if (on) {
    nb[0] = (k * ny + j) * nx + wrp(i - 1, nx); nb[1] = (k * ny + j) * nx + wrp(i + 1, nx);
    nb[2] = (k * ny + wrp(j - 1, ny)) * nx + i; nb[3] = (k * ny + wrp(j + 1, ny)) * nx + i;
    nb[4] = (wrp(k - 1, nz) * ny + j) * nx + i; nb[5] = (wrp(k + 1, nz) * ny + j) * nx + i;
  }
  T v = T(0);
  int cur = 0;
  if (init) {                                   // continue from an iterate (second visit of a W-cycle)
    if (on) { v = init[t]; buf[0][t] = v; }
    __syncthreads();
  }
  for (int s = 0; s < nu; ++s) {
    if (on) {
      if (s == 0 && !init) v = -c1 * h2 * f;
      else {
        const T* b = buf[cur];
        v = c0 * v + c1 * ((((b[nb[0]] + b[nb[1]]) + (b[nb[2]] + b[nb[3]])) + (b[nb[4]] + b[nb[5]])) - h2 * f);
      }
      buf[cur ^ 1][t] = v;
    }
    cur ^= 1;
    __syncthreads();
  }
  if (on) out[t] = v;
}

// ----------------------------------------------- the coarse levels of a cycle in ONE block (DH_MG_SUBTREE)
// A level of <= MG_SUB_MAX_CELLS cells and everything below it (16^3, 8^3, 4^3, 2^3 for power-of-two grids) is pure launch
// latency as separate kernels: a W-cycle at 512^3 visits the 16^3 level 32 times and the levels below it 2, 4, 8 times per
// visit (1600 launches of 1786).  This kernel runs that whole sub-cycle - the same operators, per cell in the same order of
// operations as the kernels above - with every level's iterate, right-hand side and Jacobi scratch in shared memory
// (3 x 4681 words for 16^3: 56 KB fp32, 112 KB fp64) and one block barrier per operator.  Level index L is a template
// parameter, so the level pointers live in registers.
constexpr int MG_SUB_MAX_CELLS = 4096;
constexpr int MG_SUB_MAX_LEV = 6;

struct MgSub {
  int nlev;
  int nx[MG_SUB_MAX_LEV], ny[MG_SUB_MAX_LEV], nz[MG_SUB_MAX_LEV];
  double h2[MG_SUB_MAX_LEV];          // h_l^2
  int nu1, nu2, gamma, nu_coarse;
  double omega;
};

template <class T>
struct MgSubMem {
  T* x[MG_SUB_MAX_LEV];               // iterate (may swap roles with s)
  T* s[MG_SUB_MAX_LEV];               // Jacobi scratch
  T* r[MG_SUB_MAX_LEV];               // right-hand side
};

template <class T>
__device__ __forceinline__ void sub_sweep(T* out, const T* in, const T* F, int nx, int ny, int nz, T c0, T c1, T h2, bool zero_in) {
  const int n = nx * ny * nz;
  for (int t = threadIdx.x; t < n; t += blockDim.x) {
    const T f = F[t];
    T o;
    if (zero_in) {
      o = -c1 * h2 * f;
    } else {
      const int i = t % nx, j = (t / nx) % ny, k = t / (nx * ny);
      const int row = (k * ny + j) * nx;
      const T sum = ((in[row + wrp(i - 1, nx)] + in[row + wrp(i + 1, nx)]) +
                     (in[(k * ny + wrp(j - 1, ny)) * nx + i] + in[(k * ny + wrp(j + 1, ny)) * nx + i])) +
                    (in[(wrp(k - 1, nz) * ny + j) * nx + i] + in[(wrp(k + 1, nz) * ny + j) * nx + i]);
      o = c0 * in[t] + c1 * (sum - h2 * f);
    }
    out[t] = o;
  }
  __syncthreads();
}

template <class T>
__device__ __forceinline__ void sub_smooth(T*& x, T*& sc, const T* F, int nx, int ny, int nz, T c0, T c1, T h2, int nu, bool from_zero) {
  for (int q = 0; q < nu; ++q) {
    sub_sweep<T>(sc, x, F, nx, ny, nz, c0, c1, h2, from_zero && q == 0);
    T* tmp = x; x = sc; sc = tmp;
  }
}

template <class T>
__device__ __forceinline__ void sub_residual_restrict(T* rc, const T* phi, const T* F, int nx, int ny, int nz, T inv_h2) {
  const int cx = nx >> 1, cy = ny >> 1, cz = nz >> 1, nc = cx * cy * cz;
  for (int t = threadIdx.x; t < nc; t += blockDim.x) {
    const int I = t % cx, J = (t / cx) % cy, K = t / (cx * cy);
    const int i = 2 * I, im = wrp(i - 1, nx), ip = wrp(i + 2, nx);
    T acc = T(0);
#pragma unroll
    for (int dk = 0; dk < 2; ++dk) {
#pragma unroll
      for (int dj = 0; dj < 2; ++dj) {
        const int j = 2 * J + dj, k = 2 * K + dk;
        const int row = (k * ny + j) * nx;
        const int rym = (k * ny + wrp(j - 1, ny)) * nx, ryp = (k * ny + wrp(j + 1, ny)) * nx;
        const int rzm = (wrp(k - 1, nz) * ny + j) * nx, rzp = (wrp(k + 1, nz) * ny + j) * nx;
        const T c0 = phi[row + i], c1 = phi[row + i + 1];
        const T s0 = ((phi[row + im] + c1) + (phi[rym + i] + phi[ryp + i])) + (phi[rzm + i] + phi[rzp + i]);
        const T s1 = ((c0 + phi[row + ip]) + (phi[rym + i + 1] + phi[ryp + i + 1])) + (phi[rzm + i + 1] + phi[rzp + i + 1]);
        acc += (F[row + i] - (s0 - T(6) * c0) * inv_h2) + (F[row + i + 1] - (s1 - T(6) * c1) * inv_h2);
      }
    }
    rc[t] = T(0.125) * acc;
  }
  __syncthreads();
}

template <class T>
__device__ __forceinline__ void sub_prolong_add(T* phi, const T* e, int nx, int ny, int nz) {
  const int cx = nx >> 1, cy = ny >> 1, cz = nz >> 1, nc = cx * cy * cz;
  for (int t = threadIdx.x; t < nc; t += blockDim.x) {
    const int I = t % cx, J = (t / cx) % cy, K = t / (cx * cy);
    const int Is[3] = {wrp(I - 1, cx), I, wrp(I + 1, cx)};
    const int Js[3] = {wrp(J - 1, cy), J, wrp(J + 1, cy)};
    const int Ks[3] = {wrp(K - 1, cz), K, wrp(K + 1, cz)};
    T x0[3][3], x1[3][3];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        const T* r = e + (Ks[a] * cy + Js[b]) * cx;
        const T m = r[Is[0]], c = r[Is[1]], p = r[Is[2]];
        x0[a][b] = T(0.75) * c + T(0.25) * m;
        x1[a][b] = T(0.75) * c + T(0.25) * p;
      }
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
      for (int dj = 0; dj < 2; ++dj) {
        const int kn = dk ? 2 : 0, jn = dj ? 2 : 0;
        const T y0c = T(0.75) * x0[1][1] + T(0.25) * x0[1][jn], y0n = T(0.75) * x0[kn][1] + T(0.25) * x0[kn][jn];
        const T y1c = T(0.75) * x1[1][1] + T(0.25) * x1[1][jn], y1n = T(0.75) * x1[kn][1] + T(0.25) * x1[kn][jn];
        const int o = ((2 * K + dk) * ny + (2 * J + dj)) * nx + 2 * I;
        phi[o] += T(0.75) * y0c + T(0.25) * y0n;
        phi[o + 1] += T(0.75) * y1c + T(0.25) * y1n;
      }
  }
  __syncthreads();
}

// one cycle on sub-level L for A x = r[L], starting from x[L] (zero if from_zero); every thread of the block takes the same path
template <class T, int L>
__device__ void sub_cycle(MgSubMem<T>& m, const MgSub& sp, bool from_zero) {
  const int nx = sp.nx[L], ny = sp.ny[L], nz = sp.nz[L], n = nx * ny * nz;
  const T c0 = (T)(1.0 - sp.omega), c1 = (T)(sp.omega / 6.0), h2 = (T)sp.h2[L];
  if (L == sp.nlev - 1) {                               // coarsest level (reading A22)
    if (sp.nu_coarse == 0) {
      if (from_zero) {
        for (int t = threadIdx.x; t < n; t += blockDim.x) m.x[L][t] = T(0);
        __syncthreads();
      }
      return;
    }
    if (n <= 32) {
      // a grid of at most one warp (2^3 for power-of-two grids): warp 0 sweeps alone with warp barriers, the block waits once
      if (threadIdx.x < 32) {
        T* a = m.x[L];
        T* b = m.s[L];
        const int t = threadIdx.x;
        const bool on = t < n;
        const int i = on ? t % nx : 0, j = on ? (t / nx) % ny : 0, k = on ? t / (nx * ny) : 0;
        const int row = (k * ny + j) * nx;
        const int n0 = row + wrp(i - 1, nx), n1 = row + wrp(i + 1, nx), n2 = (k * ny + wrp(j - 1, ny)) * nx + i,
                  n3 = (k * ny + wrp(j + 1, ny)) * nx + i, n4 = (wrp(k - 1, nz) * ny + j) * nx + i, n5 = (wrp(k + 1, nz) * ny + j) * nx + i;
        const T f = on ? m.r[L][t] : T(0);
        for (int q = 0; q < sp.nu_coarse; ++q) {
          if (on) b[t] = (from_zero && q == 0) ? -c1 * h2 * f : c0 * a[t] + c1 * ((((a[n0] + a[n1]) + (a[n2] + a[n3])) + (a[n4] + a[n5])) - h2 * f);
          __syncwarp();
          T* tmp = a; a = b; b = tmp;
        }
      }
      if (sp.nu_coarse & 1) { T* tmp = m.x[L]; m.x[L] = m.s[L]; m.s[L] = tmp; }
      __syncthreads();
      return;
    }
    sub_smooth<T>(m.x[L], m.s[L], m.r[L], nx, ny, nz, c0, c1, h2, sp.nu_coarse, from_zero);
    return;
  }
  if constexpr (L + 1 < MG_SUB_MAX_LEV) {
    sub_smooth<T>(m.x[L], m.s[L], m.r[L], nx, ny, nz, c0, c1, h2, sp.nu1, from_zero);
    if (from_zero && sp.nu1 == 0) {
      for (int t = threadIdx.x; t < n; t += blockDim.x) m.x[L][t] = T(0);
      __syncthreads();
    }
    sub_residual_restrict<T>(m.r[L + 1], m.x[L], m.r[L], nx, ny, nz, (T)(1.0 / sp.h2[L]));
    for (int v = 0; v < sp.gamma; ++v) sub_cycle<T, L + 1>(m, sp, v == 0);
    sub_prolong_add<T>(m.x[L], m.x[L + 1], nx, ny, nz);
    sub_smooth<T>(m.x[L], m.s[L], m.r[L], nx, ny, nz, c0, c1, h2, sp.nu2, false);
  }
}

template <class T>
__global__ void __launch_bounds__(1024) mg_subtree_kernel(T* x_g, const T* __restrict__ F_g, const MgSub sp, const int from_zero) {
  extern __shared__ __align__(16) unsigned char mg_sub_smem[];
  MgSubMem<T> m;
  T* q = reinterpret_cast<T*>(mg_sub_smem);
#pragma unroll
  for (int l = 0; l < MG_SUB_MAX_LEV; ++l) {
    const int n = l < sp.nlev ? sp.nx[l] * sp.ny[l] * sp.nz[l] : 0;
    m.x[l] = q; m.s[l] = q + n; m.r[l] = q + 2 * n;
    q += 3 * n;
  }
  const int n0 = sp.nx[0] * sp.ny[0] * sp.nz[0];
  for (int t = threadIdx.x; t < n0; t += blockDim.x) {
    m.r[0][t] = F_g[t];
    if (!from_zero) m.x[0][t] = x_g[t];
  }
  __syncthreads();
  sub_cycle<T, 0>(m, sp, from_zero != 0);
  for (int t = threadIdx.x; t < n0; t += blockDim.x) x_g[t] = m.x[0][t];
}

// ------------------------------------------------------------------ deterministic sums (fp64, fixed order)
constexpr int SUM_BLOCKS = 592, SUM_THREADS = 256;   // 4 blocks per SM

__device__ __forceinline__ double block_sum(double v, double* sm) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) r += sm[w];
  __syncthreads();
  return r;
}

template <class T>
__global__ void __launch_bounds__(SUM_THREADS) mg_sum_kernel(const T* __restrict__ a, size_t n, double* __restrict__ partial) {
  __shared__ double sm[SUM_THREADS / 32];
  double v = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) v += (double)a[i];
  const double r = block_sum(v, sm);
  if (threadIdx.x == 0) partial[blockIdx.x] = r;
}

// |F - A phi|^2 -> partial[b], |F|^2 -> partial[SUM_BLOCKS + b]
template <class T>
__global__ void __launch_bounds__(SUM_THREADS) mg_resnorm_kernel(const T* __restrict__ phi, const T* __restrict__ F, int nx, int ny, int nz,
                                                                 T inv_h2, double* __restrict__ partial) {
  __shared__ double sm[SUM_THREADS / 32];
  const size_t n = (size_t)nx * ny * nz;
  double vr = 0.0, vf = 0.0;
  for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(c % nx), j = (int)((c / nx) % ny), k = (int)(c / ((size_t)nx * ny));
    const size_t row = ((size_t)k * ny + j) * nx;
    const T s = ((phi[row + wrp(i - 1, nx)] + phi[row + wrp(i + 1, nx)]) +
                 (phi[((size_t)k * ny + wrp(j - 1, ny)) * nx + i] + phi[((size_t)k * ny + wrp(j + 1, ny)) * nx + i])) +
                (phi[((size_t)wrp(k - 1, nz) * ny + j) * nx + i] + phi[((size_t)wrp(k + 1, nz) * ny + j) * nx + i]);
    const double f = (double)F[c];
    const double r = f - (double)((s - T(6) * phi[c]) * inv_h2);
    vr += r * r;
    vf += f * f;
  }
  const double a = block_sum(vr, sm), b = block_sum(vf, sm);
  if (threadIdx.x == 0) { partial[blockIdx.x] = a; partial[SUM_BLOCKS + blockIdx.x] = b; }
}

// result[slot] = scale * sum_b partial[off + b]   (one thread: fixed order)
__global__ void mg_sum_finish_kernel(const double* __restrict__ partial, int off, double scale, double* __restrict__ result, int slot) {
  double s = 0.0;
  for (int b = 0; b < SUM_BLOCKS; ++b) s += partial[off + b];
  result[slot] = s * scale;
}

// out = in - result[slot]
template <class T>
__global__ void __launch_bounds__(256) mg_shift_kernel(T* out, const T* in, size_t n, const double* __restrict__ result, int slot) {
  const double m = result[slot];
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = (T)((double)in[i] - m);
}

}  // namespace

// ------------------------------------------------------------------------------------------------- context
struct dh_mg {
  int n[3];
  double h;
  int dtype;
  cudaStream_t stream;                 // the caller's stream
  cudaStream_t ls;                     // where kernels are launched: `stream`, or `cap` while a cycle is being captured
  cudaStream_t cap;                    // capture-only stream (the legacy default stream cannot be captured)
  int nu1, nu2, gamma, nu_coarse;
  double omega;
  int use_graph;
  int subtree;                         // DH_MG_SUBTREE: levels of <= 4096 cells and everything below them in one block
  int nlev;
  std::vector<int> lx, ly, lz;         // extents per level
  std::vector<void*> e, r, t;          // per level >= 1: error, right-hand side, Jacobi scratch; level 0: t only
  void* F0;                            // zero-mean copy of the right-hand side (solve)
  double* partial;                     // 2 * SUM_BLOCKS
  double* result;                      // [0] mean, [1] |r|^2, [2] |F|^2
  double* result_host;                 // pinned
  long long launches;
  // cached graph of one cycle
  cudaGraphExec_t graph;
  void* g_phi;
  const void* g_F;
  int g_key[5];
  long long g_launches;               // kernel launches inside the captured cycle
};

namespace {

size_t esize(const dh_mg* c) { return c->dtype == DH_F32 ? 4 : 8; }
size_t cells(const dh_mg* c, int l) { return (size_t)c->lx[l] * c->ly[l] * c->lz[l]; }

int mg_fail(int code, const char* where, const char* detail = "") {
  set_error(where, detail);
  return code;
}
#define MG_CUDA(call, where)                                                      \
  do {                                                                            \
    cudaError_t e_ = (call);                                                      \
    if (e_ != cudaSuccess) return mg_fail(DH_ERR_CUDA, where, cudaGetErrorString(e_)); \
  } while (0)

template <class T>
cudaError_t jacobi_launch(dh_mg* c, int l, void* out, const void* in, const void* F, bool zero_in) {
  const int nx = c->lx[l], ny = c->ly[l], nz = c->lz[l];
  const double hl = c->h * (double)(1 << l);
  const T c0 = (T)(1.0 - c->omega), c1 = (T)(c->omega / 6.0), h2 = (T)(hl * hl);
  if (nx % 4 == 0) {
    dim3 block(128), grid((nx / 4 + 127) / 128, ny, nz);
    mg_jacobi_kernel<T, 4><<<grid, block, 0, c->ls>>>((T*)out, (const T*)in, (const T*)F, nx, ny, nz, c0, c1, h2, zero_in ? 1 : 0);
  } else {
    dim3 block(128), grid((nx + 127) / 128, ny, nz);
    mg_jacobi_kernel<T, 1><<<grid, block, 0, c->ls>>>((T*)out, (const T*)in, (const T*)F, nx, ny, nz, c0, c1, h2, zero_in ? 1 : 0);
  }
  c->launches += 1;
  return cudaGetLastError();
}

// nu sweeps on level l; *pphi holds the current iterate on entry and on exit (it may be swapped with *pscratch).
template <class T>
cudaError_t smooth(dh_mg* c, int l, void** pphi, void** pscratch, const void* F, int nu, bool from_zero) {
  for (int s = 0; s < nu; ++s) {
    cudaError_t e = jacobi_launch<T>(c, l, *pscratch, *pphi, F, from_zero && s == 0);
    if (e != cudaSuccess) return e;
    void* tmp = *pphi; *pphi = *pscratch; *pscratch = tmp;
  }
  return cudaSuccess;
}

bool level_can_coarsen(int nx, int ny, int nz) { return nx % 2 == 0 && ny % 2 == 0 && nz % 2 == 0 && nx > 2 && ny > 2 && nz > 2; }

// One cycle on level l for A x = F starting from *px (zero if from_zero).  On exit *px holds the result (the pointers
// *px / *pscratch may have been swapped).
template <class T>
cudaError_t cycle_rec(dh_mg* c, int l, void** px, void** pscratch, const void* F, bool from_zero) {
  cudaError_t e;
  const int nx = c->lx[l], ny = c->ly[l], nz = c->lz[l];
  const double hl = c->h * (double)(1 << l);
  if (c->subtree && l < c->nlev - 1 && cells(c, l) <= (size_t)MG_SUB_MAX_CELLS && c->nlev - l <= MG_SUB_MAX_LEV) {
    // this level and everything below it in one block (mg_subtree_kernel)
    MgSub sp;
    sp.nlev = c->nlev - l;
    size_t words = 0;
    for (int q = 0; q < MG_SUB_MAX_LEV; ++q) {
      const bool in = q < sp.nlev;
      sp.nx[q] = in ? c->lx[l + q] : 0; sp.ny[q] = in ? c->ly[l + q] : 0; sp.nz[q] = in ? c->lz[l + q] : 0;
      const double hq = c->h * (double)(1 << (l + q));
      sp.h2[q] = hq * hq;
      if (in) words += 3 * cells(c, l + q);
    }
    sp.nu1 = c->nu1; sp.nu2 = c->nu2; sp.gamma = c->gamma; sp.nu_coarse = c->nu_coarse; sp.omega = c->omega;
    const size_t smem = words * sizeof(T);
    static bool configured[64] = {};                 // per (T, device): the opt-in to > 48 KB of dynamic shared memory
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || !configured[dev]) {
      e = cudaFuncSetAttribute((const void*)mg_subtree_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               (int)(3 * 4681 * sizeof(T)));
      if (e != cudaSuccess) return e;
      if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    // 512 threads: 1024 / 512 / 256 / 128 measured 5.03 / 4.95 / 5.06 / 5.41 ms per W-cycle at 512^3 (the block is latency bound)
    mg_subtree_kernel<T><<<1, 512, smem, c->ls>>>((T*)*px, (const T*)F, sp, from_zero ? 1 : 0);
    c->launches += 1;
    return cudaGetLastError();
  }
  if (l == c->nlev - 1) {                          // coarsest level (reading A22)
    if (cells(c, l) <= 1024 && c->nu_coarse >= 1) {
      mg_coarse_kernel<T><<<1, 1024, 0, c->ls>>>((T*)*px, from_zero ? nullptr : (const T*)*px, (const T*)F, nx, ny, nz,
                                                     (T)(1.0 - c->omega), (T)(c->omega / 6.0), (T)(hl * hl), c->nu_coarse);
      c->launches += 1;
      return cudaGetLastError();
    }
    if (from_zero && c->nu_coarse == 0) return cudaMemsetAsync(*px, 0, cells(c, l) * esize(c), c->ls);
    return smooth<T>(c, l, px, pscratch, F, c->nu_coarse, from_zero);
  }
  e = smooth<T>(c, l, px, pscratch, F, c->nu1, from_zero);
  if (e != cudaSuccess) return e;
  if (from_zero && c->nu1 == 0) {
    e = cudaMemsetAsync(*px, 0, cells(c, l) * esize(c), c->ls);
    if (e != cudaSuccess) return e;
  }
  {
    dim3 block(128), grid((nx / 2 + 127) / 128, ny / 2, nz / 2);
    mg_residual_restrict_kernel<T><<<grid, block, 0, c->ls>>>((T*)c->r[l + 1], (const T*)*px, (const T*)F, nx, ny, nz, (T)(1.0 / (hl * hl)));
    c->launches += 1;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  void* ex = c->e[l + 1];
  void* es = c->t[l + 1];
  for (int v = 0; v < c->gamma; ++v) {                 // V-cycle: one visit; W-cycle: two (Eq. C12)
    e = cycle_rec<T>(c, l + 1, &ex, &es, c->r[l + 1], v == 0);
    if (e != cudaSuccess) return e;
  }
  c->e[l + 1] = ex; c->t[l + 1] = es;                  // the two buffers may have changed roles
  {
    dim3 block(128), grid((nx / 2 + 127) / 128, ny / 2, nz / 2);
    mg_prolong_add_kernel<T><<<grid, block, 0, c->ls>>>((T*)*px, (const T*)ex, nx, ny, nz);
    c->launches += 1;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  return smooth<T>(c, l, px, pscratch, F, c->nu2, false);
}

// one cycle on the finest level, result back in the caller's phi
template <class T>
int cycle_top(dh_mg* c, void* phi, const void* F) {
  void* x = phi;
  void* s = c->t[0];
  cudaError_t e = cycle_rec<T>(c, 0, &x, &s, F, false);
  if (e != cudaSuccess) return mg_fail(DH_ERR_CUDA, "dh_mg_cycle: kernel launch", cudaGetErrorString(e));
  if (x != phi)     // an odd number of sweeps left the iterate in our scratch buffer
    MG_CUDA(cudaMemcpyAsync(phi, x, cells(c, 0) * esize(c), cudaMemcpyDeviceToDevice, c->ls), "dh_mg_cycle: copy of the iterate");
  return DH_OK;
}

// The same cycle as a CUDA graph, captured once per (phi, F, options): the coarse levels are launch bound.
template <class T>
int cycle_graph(dh_mg* c, void* phi, const void* F) {
  if (!c->use_graph) return cycle_top<T>(c, phi, F);
  const int key[5] = {c->nu1, c->nu2, c->gamma + 16 * c->subtree, c->nu_coarse, (int)(c->omega * 1e9)};
  bool same = c->graph && c->g_phi == phi && c->g_F == F;
  for (int q = 0; q < 5; ++q) same = same && c->g_key[q] == key[q];
  if (!same) {
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
    const long long before = c->launches;
    MG_CUDA(cudaStreamBeginCapture(c->cap, cudaStreamCaptureModeThreadLocal), "dh_mg_cycle: begin capture");
    c->ls = c->cap;
    const int rc = cycle_top<T>(c, phi, F);
    c->ls = c->stream;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap, &g);
    c->g_launches = c->launches - before;
    c->launches = before;
    if (rc != DH_OK) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess) return mg_fail(DH_ERR_CUDA, "dh_mg_cycle: end capture", cudaGetErrorString(e));
    e = cudaGraphInstantiate(&c->graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { c->graph = nullptr; return mg_fail(DH_ERR_CUDA, "dh_mg_cycle: graph instantiation", cudaGetErrorString(e)); }
    c->g_phi = phi; c->g_F = F;
    for (int q = 0; q < 5; ++q) c->g_key[q] = key[q];
  }
  MG_CUDA(cudaGraphLaunch(c->graph, c->stream), "dh_mg_cycle: graph launch");
  c->launches += c->g_launches;
  return DH_OK;
}

template <class T>
int mean_to_slot(dh_mg* c, const void* a, int slot) {
  const size_t n = cells(c, 0);
  mg_sum_kernel<T><<<SUM_BLOCKS, SUM_THREADS, 0, c->stream>>>((const T*)a, n, c->partial);
  mg_sum_finish_kernel<<<1, 1, 0, c->stream>>>(c->partial, 0, 1.0 / (double)n, c->result, slot);
  c->launches += 2;
  MG_CUDA(cudaGetLastError(), "dh_mg_solve: mean kernels");
  return DH_OK;
}

template <class T>
int solve_impl(dh_mg* c, const void* F, void* phi, int ncycles, double* rel_out) {
  const size_t n = cells(c, 0);
  int rc = mean_to_slot<T>(c, F, 0);                                   // reading A23: zero-mean right-hand side
  if (rc) return rc;
  mg_shift_kernel<T><<<SUM_BLOCKS, 256, 0, c->stream>>>((T*)c->F0, (const T*)F, n, c->result, 0);
  c->launches += 1;
  MG_CUDA(cudaMemsetAsync(phi, 0, n * esize(c), c->stream), "dh_mg_solve: zero initial guess");
  for (int it = 0; it < ncycles; ++it) {
    rc = cycle_graph<T>(c, phi, c->F0);
    if (rc) return rc;
  }
  rc = mean_to_slot<T>(c, phi, 0);
  if (rc) return rc;
  mg_shift_kernel<T><<<SUM_BLOCKS, 256, 0, c->stream>>>((T*)phi, (const T*)phi, n, c->result, 0);
  c->launches += 1;
  MG_CUDA(cudaGetLastError(), "dh_mg_solve: shift kernel");
  if (rel_out) {
    mg_resnorm_kernel<T><<<SUM_BLOCKS, SUM_THREADS, 0, c->stream>>>((const T*)phi, (const T*)c->F0, c->n[0], c->n[1], c->n[2],
                                                                   (T)(1.0 / (c->h * c->h)), c->partial);
    mg_sum_finish_kernel<<<1, 1, 0, c->stream>>>(c->partial, 0, 1.0, c->result, 1);
    mg_sum_finish_kernel<<<1, 1, 0, c->stream>>>(c->partial, SUM_BLOCKS, 1.0, c->result, 2);
    c->launches += 3;
    MG_CUDA(cudaMemcpyAsync(c->result_host, c->result, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "dh_mg_solve: residual copy");
    MG_CUDA(cudaStreamSynchronize(c->stream), "dh_mg_solve: synchronize");
    *rel_out = c->result_host[2] > 0.0 ? sqrt(c->result_host[1] / c->result_host[2]) : 0.0;
  }
  return DH_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

dh_mg* dh_mg_create(int nx, int ny, int nz, double h, int dtype) {
  if (nx < 2 || ny < 2 || nz < 2 || !(h > 0.0) || (dtype != DH_F32 && dtype != DH_F64)) {
    set_error("dh_mg_create: need nx, ny, nz >= 2, h > 0 and dtype DH_F32 / DH_F64", "");
    return nullptr;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    set_error("dh_mg_create: no CUDA device (there is no CPU fallback)", "");
    return nullptr;
  }
  dh_mg* c = new dh_mg();
  c->n[0] = nx; c->n[1] = ny; c->n[2] = nz; c->h = h; c->dtype = dtype; c->stream = 0; c->ls = 0; c->cap = nullptr;
  c->nu1 = 2; c->nu2 = 2; c->gamma = 1; c->nu_coarse = 64; c->omega = 2.0 / 3.0; c->use_graph = 1; c->subtree = 1;
  c->F0 = nullptr; c->partial = nullptr; c->result = nullptr; c->result_host = nullptr; c->launches = 0;
  c->graph = nullptr; c->g_phi = nullptr; c->g_F = nullptr; c->g_launches = 0;
  int x = nx, y = ny, z = nz;
  for (;;) {
    c->lx.push_back(x); c->ly.push_back(y); c->lz.push_back(z);
    if (!level_can_coarsen(x, y, z)) break;
    x /= 2; y /= 2; z /= 2;
  }
  c->nlev = (int)c->lx.size();
  c->e.assign(c->nlev, nullptr); c->r.assign(c->nlev, nullptr); c->t.assign(c->nlev, nullptr);
  const size_t es = esize(c);
  bool ok = cudaStreamCreateWithFlags(&c->cap, cudaStreamNonBlocking) == cudaSuccess && cudaMalloc(&c->F0, cells(c, 0) * es) == cudaSuccess && cudaMalloc(&c->t[0], cells(c, 0) * es) == cudaSuccess &&
            cudaMalloc((void**)&c->partial, 2 * SUM_BLOCKS * sizeof(double)) == cudaSuccess &&
            cudaMalloc((void**)&c->result, 4 * sizeof(double)) == cudaSuccess &&
            cudaMallocHost((void**)&c->result_host, 4 * sizeof(double)) == cudaSuccess;
  for (int l = 1; ok && l < c->nlev; ++l)
    ok = cudaMalloc(&c->e[l], cells(c, l) * es) == cudaSuccess && cudaMalloc(&c->r[l], cells(c, l) * es) == cudaSuccess &&
         cudaMalloc(&c->t[l], cells(c, l) * es) == cudaSuccess;
  if (!ok) {
    set_error("dh_mg_create: allocation failed", cudaGetErrorString(cudaGetLastError()));
    dh_mg_destroy(c);
    return nullptr;
  }
  return c;
}

void dh_mg_destroy(dh_mg* c) {
  if (!c) return;
  if (c->graph) cudaGraphExecDestroy(c->graph);
  if (c->cap) cudaStreamDestroy(c->cap);
  for (int l = 0; l < (int)c->t.size(); ++l) { cudaFree(c->e[l]); cudaFree(c->r[l]); cudaFree(c->t[l]); }
  cudaFree(c->F0); cudaFree(c->partial); cudaFree(c->result);
  if (c->result_host) cudaFreeHost(c->result_host);
  delete c;
}

int dh_mg_set_stream(dh_mg* c, void* stream) {
  if (!c) return mg_fail(DH_ERR_ARG, "dh_mg_set_stream: NULL context");
  c->stream = (cudaStream_t)stream;
  c->ls = c->stream;
  return DH_OK;
}

int dh_mg_set_option(dh_mg* c, int key, double v) {
  if (!c) return mg_fail(DH_ERR_ARG, "dh_mg_set_option: NULL context");
  const bool whole = v == (double)(int)v;
  switch (key) {
    case DH_MG_NU1: if (!whole || v < 0 || v > 64) return mg_fail(DH_ERR_ARG, "dh_mg_set_option: nu1 must be an integer in 0 .. 64"); c->nu1 = (int)v; break;
    case DH_MG_NU2: if (!whole || v < 0 || v > 64) return mg_fail(DH_ERR_ARG, "dh_mg_set_option: nu2 must be an integer in 0 .. 64"); c->nu2 = (int)v; break;
    case DH_MG_GAMMA: if (v != 1.0 && v != 2.0) return mg_fail(DH_ERR_ARG, "dh_mg_set_option: gamma must be 1 (V-cycle) or 2 (W-cycle)"); c->gamma = (int)v; break;
    case DH_MG_NU_COARSE: if (!whole || v < 0 || v > 4096) return mg_fail(DH_ERR_ARG, "dh_mg_set_option: nu_coarse must be an integer in 0 .. 4096"); c->nu_coarse = (int)v; break;
    case DH_MG_OMEGA: if (!(v > 0.0 && v <= 1.0)) return mg_fail(DH_ERR_ARG, "dh_mg_set_option: omega must be in (0, 1]"); c->omega = v; break;
    case DH_MG_GRAPH: c->use_graph = (v != 0.0); break;
    case DH_MG_SUBTREE: c->subtree = (v != 0.0); break;
    default: return mg_fail(DH_ERR_ARG, "dh_mg_set_option: unknown key");
  }
  return DH_OK;
}

int dh_mg_levels(const dh_mg* c) { return c ? c->nlev : 0; }

long long dh_mg_launches(const dh_mg* c) { return c ? c->launches : 0; }

int dh_mg_cycle(dh_mg* c, void* phi, const void* F) {
  if (!c || !phi || !F) return mg_fail(DH_ERR_ARG, "dh_mg_cycle: NULL argument");
  if (phi == F) return mg_fail(DH_ERR_ARG, "dh_mg_cycle: phi and F must not alias");
  return c->dtype == DH_F32 ? cycle_graph<float>(c, phi, F) : cycle_graph<double>(c, phi, F);
}

int dh_mg_solve(dh_mg* c, const void* F, void* phi, int ncycles, double* rel_residual) {
  if (!c || !phi || !F) return mg_fail(DH_ERR_ARG, "dh_mg_solve: NULL argument");
  if (phi == F) return mg_fail(DH_ERR_ARG, "dh_mg_solve: phi and F must not alias");
  if (ncycles < 0) return mg_fail(DH_ERR_ARG, "dh_mg_solve: ncycles must be >= 0");
  return c->dtype == DH_F32 ? solve_impl<float>(c, F, phi, ncycles, rel_residual) : solve_impl<double>(c, F, phi, ncycles, rel_residual);
}

int dh_mg_solve_vjp(dh_mg* c, const void* g_phi, void* g_F, int ncycles, double* rel_residual) {
  // Eqs. 46-48: A^-1 is self-adjoint, the cotangent of F is the solution of A g_F = g_phi: the same solve
  if (!c || !g_phi || !g_F) return mg_fail(DH_ERR_ARG, "dh_mg_solve_vjp: NULL argument");
  return dh_mg_solve(c, g_phi, g_F, ncycles, rel_residual);
}

}  // extern "C"
