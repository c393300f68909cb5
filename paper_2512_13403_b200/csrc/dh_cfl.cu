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
__device__ __forceinline__ float round_down(float x) { return x; }
__device__ __forceinline__ float round_down(double x) { return __double2float_rd(x); }

// ek / eth: the kinetic and thermal energy densities the recipe forms on its way (in T, with the floored density)
template <class T>
__device__ __forceinline__ void cell_speeds(T rho, T mx, T my, T mz, T E, const CflParams<T>& p, T& sx, T& sy, T& sz, bool& bad,
                                            T& ek, T& eth) {
  const T rt = (rho >= p.rho_floor) ? rho : p.rho_floor;
  const T vx = Ieee::div(mx, rt), vy = Ieee::div(my, rt), vz = Ieee::div(mz, rt);
  const T q = Ieee::add(Ieee::add(Ieee::mul(mx, mx), Ieee::mul(my, my)), Ieee::mul(mz, mz));
  ek = Ieee::mul(T(0.5), Ieee::div(q, rt));
  eth = Ieee::sub(E, ek);
  T P = Ieee::mul(p.gm1, eth);
  P = (P >= p.p_floor) ? P : p.p_floor;
  const T cs = Ieee::sqrt(Ieee::div(Ieee::mul(p.gamma, P), rt));
  const T ax = Ieee::add(abs_(vx), cs), ay = Ieee::add(abs_(vy), cs), az = Ieee::add(abs_(vz), cs);
  // the floors are compare-selects and would swallow a NaN in rho or E: test the inputs as well
  bad = bad || !(finite_(rho) && finite_(mx) && finite_(my) && finite_(mz) && finite_(E) && finite_(ax) && finite_(ay) && finite_(az));
  sx = (ax > sx) ? ax : sx;
  sy = (ay > sy) ? ay : sy;
  sz = (az > sz) ? az : sz;
}

template <class T>
__device__ __forceinline__ void cell_speeds(T rho, T mx, T my, T mz, T E, const CflParams<T>& p, T& sx, T& sy, T& sz, bool& bad) {
  T ek, eth;
  cell_speeds<T>(rho, mx, my, mz, E, p, sx, sy, sz, bad, ek, eth);
}

// Eq. 20 for one cell in the code units of reading A10, in double whatever T (reading A24); the
// operations and their order are those of cool() / cool_rate() of the cooling update, never contracted.
// (not inlined: the rare exact path is a call, so that the fp64 power function does not weigh on the registers of the sweep)
__device__ __noinline__ double cell_tcool(double rho, double mx, double my, double mz, double E, double gm1d, double lambda0, double alpha,
                                          double tmin) {
  const double q = Ieee::add(Ieee::add(Ieee::mul(mx, mx), Ieee::mul(my, my)), Ieee::mul(mz, mz));
  const double Ek = Ieee::div(Ieee::mul(0.5, q), rho);
  const double Eth = Ieee::sub(E, Ek);
  const double Tc = Ieee::div(Ieee::mul(gm1d, Eth), rho);
  const double Tpos = (Tc > 0.0) ? Tc : 0.0;
  const double rate = Ieee::mul(Ieee::mul(Ieee::mul(rho, rho), lambda0), Tc > 0.0 ? pow(Tpos, alpha) : 0.0);   // rate 0 for T <= 0, as cool_rate()
  const double t = Ieee::div(fabs(Eth), fabs(rate));
  return (rate != 0.0 && t < tmin) ? t : tmin;
}

// t_cool of Eq. 20 for the two-branch law of Eqs. 17-19 (DH_OPT_COOL_LAW = 1): |E_th| / |n_H Gamma - n_H^2 Lambda| with the rate
// of cool_rate() in double (no fp32 screen: with heating the rate has no closed log form, every cell is evaluated)
__device__ __noinline__ double cell_tcool_law(double rho, double mx, double my, double mz, double E, const Consts<double>& cd, double tmin) {
  const double q = Ieee::add(Ieee::add(Ieee::mul(mx, mx), Ieee::mul(my, my)), Ieee::mul(mz, mz));
  const double Ek = Ieee::div(Ieee::mul(0.5, q), rho);
  const double Eth = Ieee::sub(E, Ek);
  const double rate = cool_rate<double>(Eth, rho, 1.0 / rho, cd);
  const double t = Ieee::div(fabs(Eth), fabs(rate));
  return (rate != 0.0 && t < tmin) ? t : tmin;
}

// fp32 screen in front of cell_tcool (whose fp64 power function would make the pass ALU bound: 1.92 ms instead of the 0.41 ms
// the 20 B/cell take at 512^3).  Any exact t_cool already evaluated is an upper bound of the global minimum, so a cell whose
// exact value provably exceeds the warp's running minimum need not be evaluated.  The screen works in log2 on the E_kin / E_th
// the wave-speed recipe has just formed:  log2 t_cool = (1 - alpha) log2 E_th + (alpha - 2) log2 rho - log2 lambda0
// - alpha log2(gamma - 1), two MUFU.LG2 and two FMAs.  When E_th is well conditioned (|E_th| >= 2^-8 (|E| + E_kin): relative
// error of the fp32 E_th below 6e-5) and rho, E are normal fp32 numbers above the density floor, the left-hand side is within
// (1 + |1 - alpha|) 1e-4 + 1e-4 of the exact value, and lhs > lthr = log2(tmin) + log2(1 + 1e-3 (1 + |1 - alpha|)) + the constants
// proves t > tmin; a well-conditioned E_th <= 0 proves a zero rate.  Everything else (ill conditioned, out of range, NaN)
// returns true = "evaluate exactly".
// (`range_ok`: rho above the density floor and rho, S inside the fp32 range tests of speeds_may_decide, which also formed S)
template <class T>
__device__ __forceinline__ bool tcool_may_decide(T rho_, float Eth, float S, bool range_ok, float c_eth, float c_rho, float lthr) {
  const bool sure = range_ok && fabsf(Eth) >= 0.00390625f * S && S > 1e-30f;
  const float lhs = fmaf(c_eth, __log2f(Eth), c_rho * __log2f((float)rho_));
  const bool skip = sure && (Eth <= 0.0f || lhs > lthr);
  return !skip;
}

// fp32 screen in front of the wave-speed recipe (COOL sweep only; the plain reduction is HBM bound as it is).  The exact
// recipe's five IEEE divisions and square root are most of the sweep's instructions, and only cells near the maxima matter:
// a cell whose speeds are provably below exact speeds already found cannot raise the maxima.  Upper bounds from fast fp32:
// |v_a| <= |m_a| (1/rho) (1 + 1e-5);  P <= gm1 (E_th + 1e-6 (|E| + E_kin)) (the fp32 E_th is within 3e-7 (|E| + E_kin) of the
// recipe's), floored;  c_s <= sqrt(gamma P / rho) (1 + 1e-5).  Needs rho above the density floor and normal fp32 ranges;
// anything else (NaN and Inf included, so the non-finite flag is still raised by the recipe) returns true = "run the recipe".
// Also hands the fp32 E_kin / E_th to the t_cool screen.
template <class T>
__device__ __forceinline__ bool speeds_may_decide(T rho_, T mx_, T my_, T mz_, T E_, T rho_floor, float gm1f, float gammaf, float pflf,
                                                  float bx, float by, float bz, float& Ek, float& Eth, float& S, bool& sure) {
  const float rho = (float)rho_, mx = (float)mx_, my = (float)my_, mz = (float)mz_, E = (float)E_;
  const float ir = __fdividef(1.0f, rho);
  Ek = 0.5f * (mx * mx + my * my + mz * mz) * ir;
  Eth = E - Ek;
  S = fabsf(E) + Ek;
  const float Pup = fmaxf(gm1f * fmaf(1e-6f, S, Eth), pflf);
  const float cs = sqrtf(gammaf * Pup * ir) * 1.00002f;
  const float k = 1.00001f * ir;
  sure = rho_ >= rho_floor && rho > 1e-15f && rho < 1e15f && S < 1e30f;
  const bool below = fmaf(fabsf(mx), k, cs) < bx && fmaf(fabsf(my), k, cs) < by && fmaf(fabsf(mz), k, cs) < bz;
  return !(sure && below);
}

template <class T> struct Vec;
template <> struct Vec<float> { using type = float4; static constexpr int W = 4; };
template <> struct Vec<double> { using type = double2; static constexpr int W = 2; };

template <class T, bool COOL>
__global__ void __launch_bounds__(256, COOL ? 4 : 1) cfl_reduce_kernel(const CflParams<T> p, const bool guarded) {
  using V = typename Vec<T>::type;
  constexpr int W = Vec<T>::W;
  const size_t N = p.N;
  if (guarded && p.cand_cnt[1] == 0u) return;      // the candidates already hold the maxima (cfl_cand_kernel)
  T sx = T(0), sy = T(0), sz = T(0);
  double tmin = __longlong_as_double(0x7ff0000000000000ll);
  bool bad = false;
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  if constexpr (COOL) {
    // warp-uniform trip counts (the screen's threshold is shared by the warp through shuffles)
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const size_t w0 = tid - lane;
    const bool law1 = p.cd.cool_law != 0;
    const float c_eth = (float)(1.0 - p.alpha), c_rho = (float)(p.alpha - 2.0);
    // log2 of the safety factor, and the constant terms of log2 t_cool moved to the threshold's side
    const double lconst = log2(1.0 + 1e-3 * (1.0 + fabs(1.0 - p.alpha))) + log2(p.lambda0) + p.alpha * log2(p.gm1d);
    float lthr = __int_as_float(0x7f800000);     // +inf: nothing is skipped before the first exact value
    const float gm1f = (float)p.gm1, gammaf = (float)p.gamma, pflf = (float)p.p_floor * 1.000001f;
    float bx = 0.0f, by = 0.0f, bz = 0.0f;       // fp32 lower bounds of the warp's running exact maxima
    const bool vec = (N % W == 0);
    const size_t cnt = vec ? N / W : N;
    const V* r0 = reinterpret_cast<const V*>(p.U);
    const V* r1 = reinterpret_cast<const V*>(p.U + N);
    const V* r2 = reinterpret_cast<const V*>(p.U + 2 * N);
    const V* r3 = reinterpret_cast<const V*>(p.U + 3 * N);
    const V* r4 = reinterpret_cast<const V*>(p.U + 4 * N);
    for (size_t b0 = w0; b0 < cnt; b0 += nth) {
      const size_t v = b0 + lane;
      T ca[W], cb[W], cc[W], cd[W], ce[W];
      int n = 0;
      if (v < cnt) {
        if (vec) {
          const V a = __ldg(r0 + v), b = __ldg(r1 + v), c = __ldg(r2 + v), d = __ldg(r3 + v), e = __ldg(r4 + v);
#pragma unroll
          for (int l = 0; l < W; ++l) {
            ca[l] = reinterpret_cast<const T*>(&a)[l]; cb[l] = reinterpret_cast<const T*>(&b)[l]; cc[l] = reinterpret_cast<const T*>(&c)[l];
            cd[l] = reinterpret_cast<const T*>(&d)[l]; ce[l] = reinterpret_cast<const T*>(&e)[l];
          }
          n = W;
        } else {
          ca[0] = p.U[v]; cb[0] = p.U[N + v]; cc[0] = p.U[2 * N + v]; cd[0] = p.U[3 * N + v]; ce[0] = p.U[4 * N + v];
          n = 1;
        }
      }
      bool need = false, need_s = false;
#pragma unroll
      for (int l = 0; l < W; ++l)
        if (l < n) {
          float ek, eth, S;
          bool range_ok;
          need_s = need_s || speeds_may_decide<T>(ca[l], cb[l], cc[l], cd[l], ce[l], p.rho_floor, gm1f, gammaf, pflf, bx, by, bz, ek, eth, S, range_ok);
          need = need || law1 || tcool_may_decide<T>(ca[l], eth, S, range_ok, c_eth, c_rho, lthr);
        }
      if (__any_sync(full, need_s)) {      // the exact recipe for the lanes that asked, then the warp shares its maxima
        if (need_s) {
#pragma unroll
          for (int l = 0; l < W; ++l)
            if (l < n) cell_speeds<T>(ca[l], cb[l], cc[l], cd[l], ce[l], p, sx, sy, sz, bad);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          const T ox = __shfl_xor_sync(full, sx, o), oy = __shfl_xor_sync(full, sy, o), oz = __shfl_xor_sync(full, sz, o);
          sx = (ox > sx) ? ox : sx;
          sy = (oy > sy) ? oy : sy;
          sz = (oz > sz) ? oz : sz;
        }
        bx = round_down(sx); by = round_down(sy); bz = round_down(sz);
      }
      if (__any_sync(full, need)) {
        if (need) {
#pragma unroll
          for (int l = 0; l < W; ++l)
            if (l < n) tmin = law1 ? cell_tcool_law((double)ca[l], (double)cb[l], (double)cc[l], (double)cd[l], (double)ce[l], p.cd, tmin)
                               : cell_tcool((double)ca[l], (double)cb[l], (double)cc[l], (double)cd[l], (double)ce[l], p.gm1d, p.lambda0, p.alpha, tmin);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          const double ot = __shfl_xor_sync(full, tmin, o);
          tmin = (ot < tmin) ? ot : tmin;
        }
        lthr = __double2float_ru(log2(tmin) + lconst);     // tmin = +inf stays +inf; a NaN (lambda0 = 0) never skips
      }
    }
  } else if (N % W == 0) {
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
  if constexpr (COOL) {      // min over the block: shuffles, then one slot per warp (min is exact and order independent)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double ot = __shfl_xor_sync(0xffffffffu, tmin, o);
      tmin = (ot < tmin) ? ot : tmin;
    }
    __shared__ double smt[8];
    if ((threadIdx.x & 31) == 0) smt[threadIdx.x >> 5] = tmin;
    __syncthreads();
    if (threadIdx.x == 0) {
      const int nw = blockDim.x >> 5;
      for (int w = 1; w < nw; ++w) tmin = (smt[w] < tmin) ? smt[w] : tmin;
      atomicMin(p.acc + 4, (unsigned long long)__double_as_longlong(tmin));   // non-negative doubles order like their bits
    }
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
  T dt = Ieee::mul(p.cfl, best);
  const T dt_hydro = dt;
  // Eq. 21: dt <= min(dt_hydro, c_cool min_x t_cool, dt_max), the candidates compared in T (reading A24)
  const double tcool = __longlong_as_double((long long)p.acc[4]);
  p.acc[4] = 0x7ff0000000000000ull;
  if (p.cool_lim && p.c_cool > 0.0) {
    const T dc = (T)Ieee::mul(p.c_cool, tcool);
    if (dc < dt) dt = dc;
  }
  if (p.dt_max > 0.0) {
    const T dm = (T)p.dt_max;
    if (dm < dt) dt = dm;
  }
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
  p.result->tcool_min = tcool;
  p.result->dt_hydro = (double)dt_hydro;
}

template <class T>
cudaError_t launch_cfl_reduce(const CflParams<T>& p, int sm_count, cudaStream_t s) {
  constexpr int W = Vec<T>::W;
  size_t work = (p.N % W == 0) ? p.N / W : p.N;
  size_t want = (work + 255) / 256;
  int per_sm = 8;                        // 8 resident 256-thread blocks per SM
  if (p.cool_lim) {                      // the variant with the t_cool branch holds more registers: one wave of resident blocks
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cfl_reduce_kernel<T, true>, 256, 0) != cudaSuccess || per_sm < 1) per_sm = 2;
  }
  size_t cap = (size_t)sm_count * per_sm;
  int blocks = (int)(want < cap ? want : cap);
  if (blocks < 1) blocks = 1;
  if (p.cool_lim) cfl_reduce_kernel<T, true><<<blocks, 256, 0, s>>>(p, false);
  else cfl_reduce_kernel<T, false><<<blocks, 256, 0, s>>>(p, false);
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
  cfl_reduce_kernel<T, false><<<blocks, 256, 0, s>>>(p, true);    // the candidate path is never taken with the limit of Eq. 21
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
