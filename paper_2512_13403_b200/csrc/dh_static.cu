// dh_static.cu — dh_cfl_dt_static: the CFL time step of Eq. A8 for callers that must not allocate
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  No context: dh_create allocates.
//
// The existing path (dh_cfl.cu) folds block results into accumulators a context owns (cudaMalloc in dh_create).  This variant
// keeps its scratch in a file-scope device array instead:
//     g_static_scratch   DH_STATIC_SCRATCH_BYTES = 256 KiB, resident on every GPU that loads the library, until exit.
// Layout: one 32-byte record per block of the reduction {bits(max S_x), bits(max S_y), bits(max S_z), non-finite flag}.
// A block reduces a fixed chunk of DH_STATIC_CHUNK = 16384 cells, so the array bounds the grid: at most
// DH_STATIC_MAX_CELLS = 8192 x 16384 = 2^27 cells (512^3); larger grids are rejected (DH_ERR_ARG).
// Every record the finish kernel reads is written by the reduction of the same call (plain stores, no accumulation), so
// nothing has to be cleared between calls; the array keeps the last call's records.  Every call on a device shares the
// array: calls that overlap on the GPU (different streams, no dependency between them) race.
//
// The per-cell recipe (floors as compare-selects, IEEE-rounded never-contracted operations in T) and
// the epilogue dt = C min_a dx_a / max S_a are restated here; max is exact and order independent, so dt is bit-identical to
// dh_cfl_dt's whatever the shape of the reduction.
#include <cmath>
#include <cstdio>

#include "../../include/dh.h"
#include "dh_internal.cuh"

namespace dh {
void set_error(const char* where, const char* detail);   // dh_api.cu: the text dh_last_error() returns
}

#define DH_STATIC_SCRATCH_BYTES (256 * 1024)
#define DH_STATIC_CHUNK 16384
#define DH_STATIC_MAX_BLOCKS (DH_STATIC_SCRATCH_BYTES / 32)

namespace dh {
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[DH_STATIC_SCRATCH_BYTES];

struct StaticRec {
  unsigned long long s[3];
  unsigned long long bad;
};
static_assert(sizeof(StaticRec) == 32, "record size");

template <class T>
struct StaticCflParams {
  const T* U;
  size_t N;
  T gamma, gm1, rho_floor, p_floor;
  T dx[3];
  T cfl;
  StaticRec* rec;          // the device address of g_static_scratch (cudaGetSymbolAddress), never the host-side symbol
  int nblocks;
  double* out;             // DEVICE, caller-owned: {dt, max S_x, max S_y, max S_z, non-finite flag}
};

struct R {   // IEEE, non-contractable arithmetic in T
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
__device__ __forceinline__ unsigned long long sbits(float x) { return (unsigned long long)__float_as_uint(x); }
__device__ __forceinline__ unsigned long long sbits(double x) { return (unsigned long long)__double_as_longlong(x); }
__device__ __forceinline__ void sfrom(unsigned long long b, float& x) { x = __uint_as_float((unsigned)b); }
__device__ __forceinline__ void sfrom(unsigned long long b, double& x) { x = __longlong_as_double((long long)b); }
__device__ __forceinline__ float sabs(float x) { return fabsf(x); }
__device__ __forceinline__ double sabs(double x) { return fabs(x); }

template <class T>
__device__ __forceinline__ void static_cell(T rho, T mx, T my, T mz, T E, const StaticCflParams<T>& p, T& sx, T& sy, T& sz, bool& bad) {
  const T rt = (rho >= p.rho_floor) ? rho : p.rho_floor;
  const T vx = R::div(mx, rt), vy = R::div(my, rt), vz = R::div(mz, rt);
  const T q = R::add(R::add(R::mul(mx, mx), R::mul(my, my)), R::mul(mz, mz));
  const T ek = R::mul(T(0.5), R::div(q, rt));
  T P = R::mul(p.gm1, R::sub(E, ek));
  P = (P >= p.p_floor) ? P : p.p_floor;
  const T cs = R::sqrt(R::div(R::mul(p.gamma, P), rt));
  const T ax = R::add(sabs(vx), cs), ay = R::add(sabs(vy), cs), az = R::add(sabs(vz), cs);
  bad = bad || !(isfinite(rho) && isfinite(mx) && isfinite(my) && isfinite(mz) && isfinite(E) && isfinite(ax) && isfinite(ay) && isfinite(az));
  sx = (ax > sx) ? ax : sx;
  sy = (ay > sy) ? ay : sy;
  sz = (az > sz) ? az : sz;
}

// block b reduces cells [b CHUNK, min(N, (b + 1) CHUNK)) into record b (coalesced: consecutive threads, consecutive cells)
template <class T>
__global__ void __launch_bounds__(256) static_cfl_reduce_kernel(const StaticCflParams<T> p) {
  const size_t lo = (size_t)blockIdx.x * DH_STATIC_CHUNK;
  const size_t hi = (lo + DH_STATIC_CHUNK < p.N) ? lo + DH_STATIC_CHUNK : p.N;
  const size_t N = p.N;
  T sx = T(0), sy = T(0), sz = T(0);
  bool bad = false;
  for (size_t i = lo + threadIdx.x; i < hi; i += 256)
    static_cell<T>(__ldg(p.U + i), __ldg(p.U + N + i), __ldg(p.U + 2 * N + i), __ldg(p.U + 3 * N + i), __ldg(p.U + 4 * N + i), p, sx, sy, sz, bad);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const T ox = __shfl_xor_sync(0xffffffffu, sx, o), oy = __shfl_xor_sync(0xffffffffu, sy, o), oz = __shfl_xor_sync(0xffffffffu, sz, o);
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
  if (threadIdx.x == 0) {
    unsigned b = 0u;
    for (int w = 0; w < 8; ++w) {
      sx = (sm[0][w] > sx) ? sm[0][w] : sx;
      sy = (sm[1][w] > sy) ? sm[1][w] : sy;
      sz = (sm[2][w] > sz) ? sm[2][w] : sz;
      b |= smbad[w];
    }
    StaticRec r;
    r.s[0] = sbits(sx); r.s[1] = sbits(sy); r.s[2] = sbits(sz); r.bad = b ? 1ull : 0ull;
    p.rec[blockIdx.x] = r;                       // a plain store: the record holds this call's value only
  }
}

// one block: max over the records of this call (non-negative IEEE values order like their bit patterns), then dt
template <class T>
__global__ void __launch_bounds__(256) static_cfl_finish_kernel(const StaticCflParams<T> p) {
  unsigned long long m[3] = {0ull, 0ull, 0ull}, bad = 0ull;
  for (int i = threadIdx.x; i < p.nblocks; i += 256) {
    const StaticRec r = p.rec[i];
    for (int a = 0; a < 3; ++a) m[a] = r.s[a] > m[a] ? r.s[a] : m[a];
    bad |= r.bad;
  }
  __shared__ unsigned long long sm[4][256];
  for (int a = 0; a < 3; ++a) sm[a][threadIdx.x] = m[a];
  sm[3][threadIdx.x] = bad;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int t = 1; t < 256; ++t) {
      for (int a = 0; a < 3; ++a) m[a] = sm[a][t] > m[a] ? sm[a][t] : m[a];
      bad |= sm[3][t];
    }
    T S[3];
    for (int a = 0; a < 3; ++a) sfrom(m[a], S[a]);
    T best = R::div(p.dx[0], S[0]);
    for (int a = 1; a < 3; ++a) {
      const T r = R::div(p.dx[a], S[a]);
      if (r < best) best = r;
    }
    p.out[0] = (double)R::mul(p.cfl, best);
    p.out[1] = (double)S[0];
    p.out[2] = (double)S[1];
    p.out[3] = (double)S[2];
    p.out[4] = bad ? 1.0 : 0.0;
  }
}

// Set-up, once per device, with that device current: in host code `g_static_scratch` is a host-side stand-in for the device
// array, not a device address; cudaGetSymbolAddress returns the address on the current device.
static StaticRec* g_rec_of_device[64] = {};

static cudaError_t static_scratch(StaticRec** out, int* dev_out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  *dev_out = dev;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  if (!g_rec_of_device[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (e != cudaSuccess) return e;
    g_rec_of_device[dev] = (StaticRec*)ptr;
  }
  *out = g_rec_of_device[dev];
  return cudaSuccess;
}

template <class T>
static cudaError_t static_launch(const void* U, size_t N, const double* dx, double gamma, double cfl, double rho_floor, double p_floor,
                                 StaticRec* rec, double* out, cudaStream_t s) {
  StaticCflParams<T> p;
  p.U = (const T*)U; p.N = N;
  p.gamma = (T)gamma; p.gm1 = (T)(gamma - 1.0); p.rho_floor = (T)rho_floor; p.p_floor = (T)p_floor;
  for (int a = 0; a < 3; ++a) p.dx[a] = (T)dx[a];
  p.cfl = (T)cfl;
  p.rec = rec;
  p.nblocks = (int)((N + DH_STATIC_CHUNK - 1) / DH_STATIC_CHUNK);
  p.out = out;
  static_cfl_reduce_kernel<T><<<p.nblocks, 256, 0, s>>>(p);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  static_cfl_finish_kernel<T><<<1, 256, 0, s>>>(p);
  return cudaGetLastError();
}

}  // namespace
}  // namespace dh

extern "C" {

size_t dh_static_max_cells(void) { return (size_t)DH_STATIC_MAX_BLOCKS * DH_STATIC_CHUNK; }

int dh_cfl_dt_static(const void* U, int nx, int ny, int nz, int dtype, double gamma, double cfl, const double* box, double rho_floor,
                     double p_floor, double* out5_dev, void* cuda_stream) {
  using namespace dh;
  if (!U || !out5_dev) { set_error("dh_cfl_dt_static: NULL argument", ""); return DH_ERR_ARG; }
  if (nx < 4 || ny < 4 || nz < 4) { set_error("dh_cfl_dt_static: every n_a must be >= 4", ""); return DH_ERR_ARG; }
  if (dtype != DH_F32 && dtype != DH_F64) { set_error("dh_cfl_dt_static: dtype must be DH_F32 or DH_F64", ""); return DH_ERR_ARG; }
  if (!(gamma > 1.0) || !std::isfinite(gamma) || !(cfl > 0.0) || !std::isfinite(cfl) || !(rho_floor >= 0.0) || !(p_floor >= 0.0)) {
    set_error("dh_cfl_dt_static: gamma must be finite and > 1, cfl finite and > 0, the floors >= 0", "");
    return DH_ERR_ARG;
  }
  const size_t N = (size_t)nx * ny * nz;
  if (N > dh_static_max_cells()) {
    char msg[160];
    snprintf(msg, sizeof(msg), "the grid has %zu cells; the static scratch (%d bytes) holds the partial results of at most %zu", N,
             DH_STATIC_SCRATCH_BYTES, dh_static_max_cells());
    set_error("dh_cfl_dt_static", msg);
    return DH_ERR_ARG;
  }
  const int n[3] = {nx, ny, nz};
  double dx[3];
  for (int a = 0; a < 3; ++a) {
    const double L = box ? box[a] : 1.0;
    if (!(L > 0.0) || !std::isfinite(L)) { set_error("dh_cfl_dt_static: box lengths must be finite and > 0", ""); return DH_ERR_ARG; }
    dx[a] = L / n[a];
  }
  StaticRec* rec = nullptr;
  int dev = -1;
  cudaError_t e = static_scratch(&rec, &dev);
  if (e != cudaSuccess) { set_error("dh_cfl_dt_static: address of the static scratch (cudaGetSymbolAddress)", cudaGetErrorString(e)); return DH_ERR_CUDA; }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  e = dtype == DH_F32 ? static_launch<float>(U, N, dx, gamma, cfl, rho_floor, p_floor, rec, out5_dev, s)
                      : static_launch<double>(U, N, dx, gamma, cfl, rho_floor, p_floor, rec, out5_dev, s);
  if (e != cudaSuccess) { set_error("dh_cfl_dt_static: kernel launch", cudaGetErrorString(e)); return DH_ERR_CUDA; }
  return DH_OK;
}

}  // extern "C"
