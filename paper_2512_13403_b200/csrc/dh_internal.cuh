// dh_internal.cuh — context, kernel parameter blocks and launcher declarations shared by the .cu files.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "dh_math.cuh"

namespace dh {

// Parameters of one stage  out = B - frac*dt * D(U)  (Eqs. A4, A6-A7).
template <class T>
struct StageParams {
  const T* U;        // stencil input state [5][nz][ny][nx]
  const T* B;        // base state (U^n); may alias `out` (stage 2 runs in place)
  T* out;
  int nx, ny, nz;
  T inv_dx[3];       // 1 / dx_a
  T dt;              // used when dt_dev == nullptr
  const T* dt_dev;   // device-resident dt (result of the CFL kernel)
  T frac;            // 1/2 for the predictor, 1 for the corrector
  int cool;          // apply the cooling source to the result (corrector only)
  Consts<T> c;
  // CFL candidates of the NEXT step (last stage inside dh_advance only; nullptr = off): packs of the result whose
  // wave-speed estimate reaches *cand_thr are appended to cand_list (dh_cfl.cu evaluates the exact recipe on them)
  unsigned* cand_list;
  unsigned* cand_cnt;     // [0] packs appended (may exceed cand_cap: overflow = fall back to the full reduction)
  const T* cand_thr;      // [0] derated threshold for the estimate
  unsigned cand_cap;
  // z range of the launch (fused kernel only; zcnt == 0: the whole grid): planes zbeg .. zbeg + zcnt - 1, taken modulo nz
  // (dh_stream_host computes the planes whose inputs have arrived)
  int zbeg, zcnt;
  // combo != 0 (fused kernel only): out = wB B + wX U - frac dt D(U): the Shu-Osher stages of Heun / SSPRK3
  // without a pass that forms the combination first
  int combo;
  T wB, wX;
};

// Parameters of one reversed stage  out = w1 b1 + w2 b2 - frac*dt * J_D(U)^T g   (gather form).
template <class T>
struct RevParams {
  const T* U;        // primal state the stage was evaluated at
  const T* g;        // cotangent of the stage output
  const T* b1;       // optional additive terms (nullptr = none)
  const T* b2;
  T w1, w2;          // their weights (the stage weights of Heun / SSPRK3 reversed; 1 for RK2)
  T* out;
  int nx, ny, nz;
  T inv_dx[3];
  T dt;
  T frac;
  Consts<T> c;
};

// Parameters of the two launches of a fused reversed stage (dh_rev.cu).  Scratch of a z slab of SP planes: Wp [5][SP][ny][nx]
// (all cell terms except the y neighbour terms), C [5][SP][ny][nx] (encoded masked y slope cotangents) and
// Ce [5][SP][ny][ntx][2] (encoded x slope cotangents of the first and last cell of every tile row: the two x terms that
// cross a tile edge); scratch plane sp0 holds grid plane zs (faces) / z0 (gather).
template <class T>
struct RevFaceParams {
  const T* U;        // primal state the stage was evaluated at
  const T* g;        // cotangent of the stage output
  T* Wp;
  T* C;
  T* Ce;
  int nx, ny, nz;
  int zs, nout;      // first output plane and number of output planes
  int sp0, SP;
  int ntx;           // tiles per row
  size_t SPE;        // field pitch of Ce
  T coef[3];         // frac * dt / dx_a
  Consts<T> c;
};

template <class T>
struct RevGatherParams {
  const T* U;
  const T* Wp;
  const T* C;
  const T* Ce;
  const T* b1;       // optional additive terms (nullptr = none)
  const T* b2;
  T w1, w2;          // their weights
  T* out;
  int nx, ny, nz;
  int z0, nplanes;   // planes z0 .. z0 + nplanes - 1 (all inside [0, nz))
  int sp0, SP;
  int ntx;
  size_t SPE;
  Consts<T> c;
};

// result block of the CFL reduction (device + pinned host mirror); all slots 8 bytes wide
struct CflResult {
  double smax[3];    // T values widened
  double dt;         // T value widened
  unsigned long long nonfinite;
  double tcool_min;  // min_x t_cool(x) of Eq. 20 (+inf if the limit of Eq. 21 was not evaluated)
  double dt_hydro;   // the Eq. A8 value before the other candidates of Eq. 21 (T value widened)
};

template <class T>
struct CflParams {
  const T* U;
  size_t N;
  T gamma, gm1, rho_floor, p_floor;
  T dx[3];
  T cfl;
  unsigned long long* acc;   // [0..2] running max (bit pattern of T, zero-extended), [3] non-finite flag,
                             // [4] running min of t_cool (bit pattern of a non-negative double; armed with +inf)
  // Eq. 21: cool_lim != 0 makes the reduction evaluate Eq. 20 per cell (in double, reading A24)
  int cool_lim;
  double gm1d, lambda0, alpha, c_cool, dt_max;
  Consts<double> cd;         // the cooling law in double (DH_OPT_COOL_LAW = 1: its table pointer is the double copy)
  T* dt_dev;                 // dt in T for the stage kernels
  CflResult* result;         // device copy of the result block
  // candidate path (all nullptr = plain reduction): see StageParams
  const unsigned* cand_list;
  unsigned* cand_cnt;        // [0] packs appended by the last stage, [1] "the full reduction is needed" flag
  T* cand_thr;               // [0] derated threshold for the estimate, [1] theta = 0.97 min_a S_a of the last dt
  unsigned cand_cap;
  unsigned long long* cand_stats;   // [0] candidate passes, [1] fallbacks to the full reduction, [2] packs evaluated
};

struct Ctx {
  int nx, ny, nz, dtype;
  size_t N;
  double gamma, cfl, L[3];
  int cooling, kernel, limiter, riemann, integrator;
  int cool_mode, cool_nsub;    // DH_OPT_COOL_MODE (0 Euler sub-cycled, 1 trapezoid, 2 masked per cell), DH_OPT_COOL_NSUB
  int cool_law;                // DH_OPT_COOL_LAW (0 power law, 1 the two-branch law of Eqs. 17-19)
  double t_switch, lambda1, alpha1, lambda2, alpha2, gamma0, f_sub;
  void* tab_dev;               // the table in the array dtype (log2 Lambda at nodes equally spaced in log2 T), 256 slots
  double* tab_dev_d;           // the same in double (cooling-time limit, table gradient)
  double* tab_part;            // per-block partial sums of the table gradient
  int ntab;
  double tab_log10t0, tab_dlog10t;
  double c_cool, dt_max;       // DH_OPT_C_COOL, DH_OPT_DT_MAX (Eq. 21; 0 = candidate off)
  double lambda0, alpha, t_floor, rho_floor, p_floor;
  cudaStream_t stream;
  int sm_count;
  int device;              // the device the context was created on; every entry point checks it is current
  void* Us;                    // U* scratch (always)
  void* gs;                    // cotangent of U* (first VJP)
  void* Ub;                    // base-state combination (Heun / SSPRK3); reused as the scaled cotangent in their VJP
  void* Uc;                    // second stage state of SSPRK3
  void* ga;                    // cotangent of the first stage state (SSPRK3 VJP)
  void* U1;                    // pre-cooling state, cooling VJP only
  void* g1;                    // cotangent of U1, cooling VJP only
  void* grav_phi;              // self-gravity (dh_step_gravity*): potential, right-hand side / its cotangent, the three acceleration
  void* grav_F;                //   cotangents, the post-hydro state and the cotangent handed to the hydro VJP
  void* grav_gb;
  void* grav_U1;
  void* grav_g1;
  void* Uhost_dev;             // device state for the HOST entry points
  void* Uhost_dev2;            // dh_stream_host: the second device state (steps alternate between the two)
  cudaStream_t h2d_stream, d2h_stream;   // dh_stream_host: one stream per link direction (non-blocking, created on first use)
  cudaEvent_t* ev_slab;        // dh_stream_host: [3][ev_n] slab arrived / slab computed / slab written back
  int ev_n;
  int stream_slab_opt;         // DH_OPT_STREAM_SLAB (0 = automatic)
  void* gA;                    // device cotangent buffers for dh_step_vjp_host
  void* gB;
  void* rev_scratch;           // 20 words per cell of a z slab (+2 planes), fused reverse stages
  int rev_slab;                // planes per slab the scratch was sized for
  int rev_words;               // scratch words per cell it was sized for (depends on the limiter)
  int rev_slab_opt;            // DH_OPT_REV_SLAB (0 = automatic)
  void* adj_states;            // dh_adjoint: checkpoints, one segment of states, one cotangent
  size_t adj_count;            // states allocated there
  double* adj_dts_dev;         // dh_adjoint: dt sequence (device, T widened by the CFL epilogue)
  double* adj_dts_host;        // pinned mirror
  int adj_dts_cap;
  unsigned* cand_list;         // dh_advance: CFL candidates pushed by the last stage (packs), see StageParams
  unsigned* cand_cnt;
  void* cand_thr;
  unsigned long long* cand_stats;
  unsigned cand_cap;
  int cand_ok;                 // the last stage launched did push candidates for the state it wrote
  int fuse_cfl;                // DH_OPT_FUSE_CFL
  unsigned long long* acc;     // device accumulators of the CFL reduction
  void* dt_dev;                // device dt (T)
  CflResult* result_dev;
  CflResult* result_host;      // pinned
  unsigned long long launches;
  // per-kernel event timing (dh_profile_enable / dh_profile_read)
  int prof_on;
  struct ProfRec* prof;        // pending (kind, start, stop) records
  int prof_n, prof_cap;
};

struct ProfRec {
  int kind;
  cudaEvent_t a, b;
};

size_t elem_size(const Ctx* c);

// launchers (each returns the cudaError_t of the launch)
template <class T> cudaError_t launch_stage_naive(const StageParams<T>& p, int limiter, int riemann, cudaStream_t s);
template <class T> cudaError_t launch_stage_fused2(const StageParams<T>& p, int limiter, int riemann, int sm_count, cudaStream_t s, bool* supported);
template <class T, int RS, bool COMBO> cudaError_t launch_stage_fused2_rs(const StageParams<T>& p, int limiter, int sm_count, cudaStream_t s, bool* supported);
template <class T> cudaError_t launch_rev_naive(const RevParams<T>& p, int limiter, int riemann, cudaStream_t s);
template <class T> cudaError_t launch_rev_faces(const RevFaceParams<T>& p, int limiter, int riemann, int sm_count, cudaStream_t s);
int rev_scratch_words(int limiter);
template <class T> cudaError_t launch_rev_gather(const RevGatherParams<T>& p, int limiter, cudaStream_t s);
template <class T> cudaError_t launch_cool_fwd(T* U, size_t N, T dt, const T* dt_dev, const Consts<T>& c, cudaStream_t s);
template <class T> cudaError_t launch_cool_vjp(const T* U1, const T* g, T* gout, size_t N, T dt, const Consts<T>& c, cudaStream_t s);
template <class T> cudaError_t launch_cool_table_vjp(const T* U1, const T* g, size_t N, T dt, const Consts<T>& c, double* part, double* gtab, cudaStream_t s);
int cool_table_blocks();
// self-gravity source (dh_gravity.cu)
template <class T> cudaError_t launch_grav_rhs(const T* rho, T* F, size_t N, T four_pi_g, cudaStream_t s);
template <class T> cudaError_t launch_grav_rhs_vjp(const T* gF, T* grho, size_t N, T four_pi_g, cudaStream_t s);
template <class T> cudaError_t launch_grav_source(T* U, const T* phi, int nx, int ny, int nz, const double dx[3], T dt, const T* dt_dev, cudaStream_t s);
template <class T> cudaError_t launch_grav_source_vjp(const T* U, const T* phi, const T* gout, T* gin, T* gb, T* gphi, int nx, int ny, int nz,
                                                      const double dx[3], T dt, cudaStream_t s);
template <class T> cudaError_t launch_lincomb(T* out, T a, const T* X, T b, const T* Y, size_t n, int sm_count, cudaStream_t s);
template <class T> cudaError_t launch_cfl_reduce(const CflParams<T>& p, int sm_count, cudaStream_t s);
template <class T> cudaError_t launch_cfl_candidates(const CflParams<T>& p, int sm_count, cudaStream_t s);   // candidates, then the guarded full pass
template <class T> cudaError_t launch_cfl_finish(const CflParams<T>& p, cudaStream_t s);

}  // namespace dh
