/* dh.h — C ABI of the B200-native (sm_100a) hot path of arxiv/paper_2512_13403 ("diffhydro").
 *
 * One explicit time step of the 3D compressible Euler finite-volume update on a uniform periodic
 * Cartesian grid, and its discrete adjoint.  The operation is the paper's pure step
 *     U^{n+1} = H(U^n)                                   (Eq. 1)
 * on global dense field arrays, with a separate time-step query (
 * Eq. A8) and a vector-Jacobian product in which dt is data.
 *
 * Scheme (App. A; the readings of silent points are listed in DESIGN.md):
 *   W = (rho, v, P), P = (gamma-1)(E - rho|v|^2/2)        (Eq. 2)
 *   dW_i = minmod(W_{i+1}-W_i, W_i-W_{i-1}),  W^L_{i+1/2} = W_i + dW_i/2,
 *   W^R_{i+1/2} = W_{i+1} - dW_{i+1}/2                    (Eqs. A1-A2)
 *   F = HLLC(W^L, W^R) with S_L = min(v_L-c_L, v_R-c_R), S_R = max(v_L+c_L, v_R+c_R)
 *                                                         (Eq. A3)
 *   D(U)_i = sum_a (F_{a,i+1/2} - F_{a,i-1/2}) / dx_a     (Eq. A4)
 *   U* = U^n - dt/2 D(U^n);  U^{n+1} = U^n - dt D(U*)     (Eqs. A6-A7, unsplit)
 *   optional cooling of E after the update                (Eqs. 23-24)
 *   dt = C_CFL min_a dx_a / max_cells(|v_a| + c_s)        (Eq. A8)
 *
 * ARRAYS.  A state is ONE contiguous array [5][nz][ny][nx] of T (float for DH_F32, double for
 * DH_F64): field f in {0: rho, 1: rho*v_x, 2: rho*v_y, 3: rho*v_z, 4: E},
 * x fastest, no ghost cells, periodic in x, y and z.  Unless a function says HOST, every array
 * pointer is a DEVICE pointer (e.g. torch.Tensor.data_ptr()), at least 16-byte aligned.  The caller
 * owns all arrays; the library neither frees nor retains them beyond the call (work is ordered on the
 * context's stream).  The library owns its scratch (one state for U*, further states allocated
 * lazily on the first VJP, reduction slots) and frees it in dh_destroy.
 *
 * GRID.  Unit box by default: dx_a = L_a / n_a with L = (1,1,1) (settable).  n_a >= 4.
 *
 * ERRORS.  Functions return DH_OK or a negative code; dh_last_error() gives a message for the last
 * failure on the calling thread.  No function falls back to a CPU path: if no CUDA device / kernel
 * image for sm_100 is available the call fails with DH_ERR_CUDA.
 *
 * THREADS.  One context per stream; a context is not re-entrant.
 */
#ifndef DH_H_
#define DH_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dh_ctx dh_ctx;

enum { DH_F32 = 0, DH_F64 = 1 };

enum {
  DH_OK = 0,
  DH_ERR_ARG = -1,       /* bad argument (NULL, n_a < 4, dt <= 0 or non-finite, unknown option ...) */
  DH_ERR_CUDA = -2,      /* a CUDA runtime call or kernel launch failed */
  DH_ERR_ALLOC = -3,     /* device or pinned-host allocation failed */
  DH_ERR_NONFINITE = -4  /* dh_cfl_dt: a NaN/Inf input or wave speed was found */
};

/* Keys of dh_set_option / dh_get_option.  Values are doubles; flags are 0 / 1. */
enum {
  DH_OPT_CFL = 0,        /* C_CFL of Eq. A8, default 0.4 */
  DH_OPT_LX = 1,         /* box lengths, default 1; dx_a = L_a / n_a */
  DH_OPT_LY = 2,
  DH_OPT_LZ = 3,
  DH_OPT_COOLING = 4,    /* 0 (default) / 1: E_th <- max(E_floor(rho), E_th - rho^2 Lambda0 T^alpha dt) after stage 2
                            (other integrators of the source: DH_OPT_COOL_MODE, DH_OPT_COOL_NSUB) */
  DH_OPT_LAMBDA0 = 5,    /* default 1e-3 */
  DH_OPT_ALPHA = 6,      /* default 0.5 */
  DH_OPT_T_FLOOR = 7,    /* default 0.01; E_floor = rho T_floor / (gamma-1) (Eq. 24 with R = 1) */
  DH_OPT_RHO_FLOOR = 8,  /* floors used only inside the primitive conversion, default 1e-10 */
  DH_OPT_P_FLOOR = 9,
  DH_OPT_KERNEL = 10,    /* 0 (default): fused z-sweep stage kernel, 2x2 cells per thread; 1: one-thread-per-cell gather
                            kernels (same arithmetic, kept for cross-checking and as the fallback for odd nx) */
  DH_OPT_LIMITER = 11,   /* 0 minmod (default), 1 van Leer, 2 MC */
  DH_OPT_REV_SLAB = 12,  /* planes per z slab of the fused reverse stages' scratch (10 words per cell of a slab, 15 with the
                            van Leer / MC limiters, plus a thin array of tile-edge terms);
                            0 (default): as many as fit in min(48 GiB, 70 % of the free device memory) */
  DH_OPT_INTEGRATOR = 13,/* 0 (default): the predictor / corrector of Eqs. A6-A7;
                            1: Heun's RK2  U1 = U - dt D(U);  U' = 1/2 U + 1/2 (U1 - dt D(U1));
                            2: SSPRK3  U1 = U - dt D(U);  U2 = 3/4 U + 1/4 (U1 - dt D(U1));
                               U' = 1/3 U + 2/3 (U2 - dt D(U2)).  Same stage kernels; the convex combinations are
                               formed by a streaming kernel (DH_K_LINCOMB); dh_step_vjp / dh_adjoint follow the option */
  DH_OPT_FUSE_CFL = 14,  /* 1 (default) / 0: inside dh_advance, from the second step on, the last stage of a step appends the
                            packs of its result whose estimated wave speed reaches 0.97 x the previous maximum to a list,
                            and the next dt comes from the exact recipe on that list (the full reduction runs only
                            when the list cannot settle the maxima).  dt and the states are bit-identical either way */
  DH_OPT_RIEMANN = 15,   /* Riemann flux at the faces, all with the wave speeds of Eq. A3: 0 HLLC (default),
                            1 two-wave HLL, 2 Rusanov / local Lax-Friedrichs.  Forward: the fused stage kernel;
                            dh_step_vjp / dh_adjoint with 1 or 2: the one-thread-per-cell gather kernels */
  DH_OPT_COOL_MODE = 16, /* integrator of the cooling source: 0 (default) the Euler update with floor of Eq. 23,
                            sub-cycled DH_OPT_COOL_NSUB times; 1 the trapezoid of Eq. 22 with T^pred from the Euler-predicted,
                            floored energy (reading A20); 2 either of them per cell (DH_OPT_COOL_FSUB).  (0, N_sub = 1) with
                            the power law runs in the last stage's epilogue; the others as one streaming pass over the
                            finished state (DH_K_COOL) */
  DH_OPT_COOL_NSUB = 17, /* N_sub of Eq. 23: integer in 1 .. 64, default 1; substeps dt / N_sub, rate and floor every substep */
  DH_OPT_C_COOL = 18,    /* c_cool of Eq. 21, finite >= 0, default 0 = no cooling-time limit.  With DH_OPT_COOLING = 1 and
                            c_cool > 0 every CFL pass (dh_cfl_dt, dh_cfl_dt_async, dh_advance, dh_adjoint, dh_run_host) also reduces
                            min_x t_cool(x) of Eq. 20 in the same sweep over the five fields (no extra HBM traffic) and returns
                            dt = min(dt_hydro, c_cool min_x t_cool, dt_max).  Code units of DH_OPT_COOLING: n_H = rho, Gamma = 0,
                            t_cool = |E_th| / (rho^2 Lambda0 max(T,0)^alpha), formed in fp64 whatever the dtype; cells with zero
                            rate do not count; the candidates are compared in the dtype (reading A24).  dt is
                            bit-identical to Eq. A8 whenever the hydro candidate is the smallest */
  DH_OPT_DT_MAX = 19,    /* Delta t_max of Eq. 21, finite >= 0, default 0 = none; applies with or without cooling */
  DH_OPT_COOL_LAW = 20,  /* 0 (default): Lambda = Lambda0 T^alpha, Gamma = 0; 1: the two-branch law of Eqs. 17-19:
                            T < t_switch: Lambda = lambda1 T^alpha1 + lambda2 T^alpha2 (Eq. 18) and uniform heating n_H Gamma0;
                            T >= t_switch: Lambda_CIE(T) by linear interpolation in log T - log Lambda of the table given to
                            dh_set_cooling_table (Eq. 19; end values held outside), no heating.  Code units n_H = rho, T = P / rho.
                            Needs a table first.  The update runs as the streaming pass DH_K_COOL; Eq. 20's t_cool follows the law */
  DH_OPT_T_SWITCH = 21,  /* the 10^4 K of Eq. 17 in code units, > 0, default 1 */
  DH_OPT_LAMBDA1 = 22,   /* Eq. 18, >= 0, default 0 */
  DH_OPT_ALPHA1 = 23,    /* default 1 */
  DH_OPT_LAMBDA2 = 24,   /* >= 0, default 0 */
  DH_OPT_ALPHA2 = 25,    /* default 0.5 */
  DH_OPT_GAMMA0 = 26,    /* Gamma_0 of PAPER.md:286, 294, >= 0, default 0 */
  DH_OPT_STREAM_SLAB = 28, /* planes per z slab of dh_stream_host's copies, integer >= 0; 0 (default): nz / 32, at least 8 */
  DH_OPT_COOL_FSUB = 27, /* DH_OPT_COOL_MODE = 2 (the masked per-cell choice of PAPER.md:342): a cell takes the sub-cycled update
                            of Eq. 23 (DH_OPT_COOL_NSUB substeps) when dt |Edot(T^n)| > f_sub |E_th^n|, else the trapezoid of
                            Eq. 22 (reading A26); > 0, default 0.1 */
  DH_OPT_COUNT_
};

/* Create a context for an nx x ny x nz periodic grid, adiabatic index gamma, dtype DH_F32/DH_F64, on the
 * current CUDA device.  Allocates the U* scratch state.  Returns NULL on failure (see dh_last_error). */
dh_ctx* dh_create(int nx, int ny, int nz, double gamma, int dtype);

/* Free the context and everything it owns.  NULL is allowed. */
void dh_destroy(dh_ctx* ctx);

/* Use `cuda_stream` (a cudaStream_t) for all subsequent work of this context.  Default: stream 0. */
int dh_set_stream(dh_ctx* ctx, void* cuda_stream);

int dh_set_option(dh_ctx* ctx, int key, double value);
int dh_get_option(const dh_ctx* ctx, int key, double* value_out);

/* The table of Eq. 19 for DH_OPT_COOL_LAW = 1: log10_lambda[n] (HOST, copied) = log10 Lambda_CIE at the
 * nodes log10 T = log10_t0 + k dlog10_t, k = 0 .. n-1, 2 <= n <= 256, dlog10_t > 0.  Synchronises the context's stream.
 * DH_ERR_ARG on a non-finite value or a bad size. */
int dh_set_cooling_table(dh_ctx* ctx, const double* log10_lambda, int n, double log10_t0, double dlog10_t);

/* Gradient with respect to the cooling table itself: for the step U^n -> U^{n+1} of dh_step at this dt and
 * the cotangent gU_out = dL/dU^{n+1} (DEVICE, like dh_step_vjp), gtab_out[n] (HOST) = dL / d log10_lambda[k].  The
 * pre-cooling state is recomputed; per-block partial sums are added in a fixed order.  Synchronises the stream.
 * Needs DH_OPT_COOLING = 1 and DH_OPT_COOL_LAW = 1. */
int dh_cool_table_vjp(dh_ctx* ctx, const void* U, double dt, const void* gU_out, double* gtab_out);

/* CFL time step, Eq. A8: one block-reduced max-wavespeed kernel over the 5 fields, then
 * dt = C * min_a(dx_a / S_a) formed on the device in T with IEEE-rounded, non-contracted operations, so
 * that it is bit-identical to the same recipe evaluated on a CPU.  U: DEVICE, read only.
 * dt_out: HOST; receives the T value widened exactly.  Synchronises the stream (the only host sync of
 * the path).  Returns DH_ERR_NONFINITE (and leaves *dt_out untouched) if any input or speed is NaN/Inf. */
int dh_cfl_dt(dh_ctx* ctx, const void* U, double* dt_out);

/* Eq. A8 for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): NO context (dh_create allocates) and no cudaMalloc / cudaFree / allocating library call inside.  The scratch of the
 * reduction (one 32-byte record of block maxima per 16384 cells) lives in a file-scope device array of 256 KiB that every GPU
 * loading the library holds until exit, so the grid is limited to dh_static_max_cells() = 2^27 cells (512^3); larger grids return
 * DH_ERR_ARG with a message saying so.  Same per-cell recipe and epilogue as dh_cfl_dt: dt is bit-identical to it.
 *   U:         DEVICE, read only, [5][nz][ny][nx] of `dtype` (DH_F32 / DH_F64).
 *   box:       HOST, the three box lengths, or NULL for 1, 1, 1.   gamma > 1, cfl > 0, floors >= 0 (dh_create's defaults: 1e-10).
 *   out5_dev:  DEVICE, caller-owned, 5 doubles: dt (the T value widened), max S_x, max S_y, max S_z, 1.0 if a NaN / Inf input
 *              or wave speed was seen (dt is then meaningless), else 0.0.
 *   cuda_stream: the stream both kernels are launched on (NULL = the default stream).  Asynchronous; nothing is synchronised.
 * The device array is shared by every call on that GPU and keeps the last call's records (each call overwrites the records it
 * reads, nothing has to be cleared): calls that overlap on the GPU, e.g. on two streams without a dependency, race.  The array's
 * device address is looked up once per device (cudaGetSymbolAddress, with that device current, at the first call there). */
int dh_cfl_dt_static(const void* U, int nx, int ny, int nz, int dtype, double gamma, double cfl, const double* box, double rho_floor,
                     double p_floor, double* out5_dev, void* cuda_stream);
size_t dh_static_max_cells(void);

/* min_x t_cool(x), Eq. 20, for the cooling parameters of the context (DH_OPT_LAMBDA0 / DH_OPT_ALPHA; DH_OPT_COOLING
 * need not be on): one pass of the CFL reduction kernel with the cooling-time branch.  U: DEVICE, read only.
 * tcool_min_out: HOST (+inf if no cell cools).  dt_hydro_out: HOST or NULL, the Eq. A8 value of the same pass.  Like dh_cfl_dt
 * it synchronises the stream, leaves the dt of Eq. 21 in the context's device slot, and returns DH_ERR_NONFINITE on NaN/Inf. */
int dh_cool_tmin(dh_ctx* ctx, const void* U, double* tcool_min_out, double* dt_hydro_out);

/* One step in place, U^n -> U^{n+1} (stage 1 into the library's U* scratch, stage 2 back into U, cooling
 * in the stage-2 epilogue if enabled).  U: DEVICE, read and overwritten.  dt > 0 finite.  Asynchronous on
 * the context's stream. */
int dh_step(dh_ctx* ctx, void* U, double dt);

/* Same, with dt taken from the device-resident result of the last dh_cfl_dt_async / dh_cfl_dt on this
 * context (no host round trip). */
int dh_step_devdt(dh_ctx* ctx, void* U);

/* Eq. A8 without the host read-back: leaves dt in the context's device slot for dh_step_devdt.
 * Non-finite detection is deferred to dh_poll_status. */
int dh_cfl_dt_async(dh_ctx* ctx, const void* U);

/* Synchronise the stream and report (dt of the last CFL, non-finite flag -> DH_ERR_NONFINITE). */
int dh_poll_status(dh_ctx* ctx, double* dt_out);

/* nsteps x (Eq. A8 time step + RK2 step) in place, everything on the device: per step the CFL reduction, its
 * one-thread dt epilogue, the predictor and the corrector; dt never visits the host.  (Reducing the wave speeds of
 * U^{n+1} inside the corrector instead was built and measured: the estimate-then-exact candidate test costs the
 * corrector more than the 20 B/cell pass it saves.)
 * U: DEVICE.  dt_last_out: HOST or NULL; if non-NULL the call synchronises and reports the last dt / a non-finite
 * state like dh_poll_status, otherwise it is asynchronous and dh_poll_status may be called later. */
int dh_advance(dh_ctx* ctx, void* U, int nsteps, double* dt_last_out);

/* Vector-Jacobian product of the full step (dt held constant):
 *   gU_in = (dU^{n+1}/dU^n)^T gU_out   evaluated at U = U^n (the PRE-step state) and dt.
 * Nothing is stored by dh_step: U* is recomputed, then the two stages are reversed by gather-form kernels
 * (no atomics; deterministic).  U, gU_out: DEVICE, read only.  gU_in: DEVICE, overwritten; must not alias
 * U or gU_out.  Asynchronous on the context's stream. */
int dh_step_vjp(dh_ctx* ctx, const void* U, double dt, const void* gU_out, void* gU_in);

/* Adjoint of `nsteps` steps with sparse checkpoints and recomputation of short segments (§2.3;
 * SURVEY.md §8(f) item 1).  Forward: U_0 -> U_n in place, dt_k from Eq. A8 before every step (device resident), every
 * `every`-th state and all dt_k kept.  Reverse: walking the segments backwards, the states of a segment are recomputed
 * from its checkpoint and dh_step_vjp is applied step by step with dt_k held constant.
 *   U:  DEVICE, in: U_0, out: U_n.      gU: DEVICE, in: dL/dU_n, out: dL/dU_0 (overwritten); must not alias U.
 *   every >= 1: checkpoint spacing; the library allocates ceil(nsteps / every) + every + 1 states on first use
 *   (about 2 sqrt(nsteps) states for every ~ sqrt(nsteps)) and keeps them until dh_destroy.
 *   dts_out: HOST array of nsteps doubles, or NULL.
 * Synchronises the stream once (after the forward sweep, to fetch the dt sequence); returns DH_ERR_NONFINITE if a
 * CFL reduction of the forward sweep found a non-finite state. */
int dh_adjoint(dh_ctx* ctx, void* U, void* gU, int nsteps, int every, double* dts_out);

/* HOST-buffer entry points (used for end-to-end measurements): U_host is a HOST array (pinned memory gives
 * asynchronous copies) of the same layout.  The library copies it to a device state it owns, runs
 * `nsteps` x (CFL dt + step) with the device-resident dt, copies the result back and synchronises.
 * dt_last_out (HOST, may be NULL) receives the last dt. */
int dh_run_host(dh_ctx* ctx, void* U_host, int nsteps, double* dt_last_out);

/* A state that LIVES in host memory: `nsteps` x (CFL dt + step), every step reading its input from U_host and writing its
 * result back there (the host sees every intermediate state; 2 x state bytes cross the link per step).  Same steps as
 * dh_advance (Eqs. A4-A8): U_host ends bit-identical to dh_run_host called nsteps times with one step each.
 *   U_host: HOST, in/out, same layout; pinned memory (cudaHostAlloc / cudaHostRegister) is what makes the copies
 *           asynchronous.  It must not be written by the caller during the call.
 * The state moves in z slabs of DH_OPT_STREAM_SLAB planes on two copy streams the context owns, one per link direction:
 * the write-back of step n, slab k is followed by the read of step n+1, slab k, the predictor of a step runs over the planes
 * whose neighbours have arrived, the corrector slab by slab ahead of its write-back; dt of step n+1 comes from the device copy
 * of step n's result.  In the steady state both directions are busy and a step costs max(H2D, D2H) instead of their sum plus the
 * kernels.  The library holds two device states.  Heun / SSPRK3, the cooling integrators that run as a pass of their own and
 * DH_OPT_KERNEL = 1 compute whole steps between the slab-wise copies.  Synchronises; dt_last_out as in dh_run_host. */
int dh_stream_host(dh_ctx* ctx, void* U_host, int nsteps, double* dt_last_out);

/* HOST-buffer VJP: copies U and gU_out in, runs dh_step_vjp, copies gU_in out, synchronises. */
int dh_step_vjp_host(dh_ctx* ctx, const void* U_host, double dt, const void* gU_out_host, void* gU_in_host);

/* Number of kernel launches issued by this context since creation (bench.py's gpu_launches). */
unsigned long long dh_launch_count(const dh_ctx* ctx);

/* Per-kernel device timing (used by bench.py for the roofline of each kernel).  While enabled, every kernel
 * launch of this context is bracketed by a pair of CUDA events on the context's stream.  dh_profile_read
 * synchronises the stream and ADDS the elapsed milliseconds / launch counts recorded since the last read into
 * ms_out[DH_K_COUNT_] / launches_out[DH_K_COUNT_] (HOST arrays the caller zeroes; either may be NULL). */
enum {
  DH_K_CFL_REDUCE = 0,   /* max-wavespeed reduction, Eq. A8: the full pass over the five fields (20 B/cell) */
  DH_K_CFL_FINISH = 1,   /* one-thread dt epilogue */
  DH_K_STAGE1 = 2,       /* predictor stage  U* = U^n - dt/2 D(U^n) */
  DH_K_STAGE2 = 3,       /* corrector stage  U^{n+1} = U^n - dt D(U*) (+ cooling) */
  DH_K_REV2 = 4,         /* reverse corrector */
  DH_K_REV1 = 5,         /* reverse predictor */
  DH_K_COOL_VJP = 6,     /* pointwise cooling adjoint */
  DH_K_LINCOMB = 7,      /* out = a X + b Y: base states / scaled cotangents of Heun and SSPRK3 */
  DH_K_COOL = 8,         /* in-place cooling pass of DH_OPT_COOL_MODE = 1 / DH_OPT_COOL_NSUB > 1 */
  DH_K_CFL_CAND = 9,     /* dh_advance, steps 2..: exact recipe on the listed candidate packs + the guarded full pass
                            (which returns at once unless the list cannot settle the maxima: dh_cfl_stats counts those) */
  DH_K_COUNT_ = 10
};
int dh_profile_enable(dh_ctx* ctx, int on);
int dh_profile_read(dh_ctx* ctx, double* ms_out, unsigned long long* launches_out);

/* Counters of the CFL candidate path of dh_advance (DH_OPT_FUSE_CFL) since dh_create, copied to the HOST array
 * out[3] after a synchronize of the context's stream: out[0] = dt's taken from a candidate list, out[1] = of those,
 * the ones that fell back to the full reduction (list overflow, or a maximum below the threshold), out[2] = packs
 * evaluated with the exact recipe.  All zero before the first dh_advance of more than one step. */
int dh_cfl_stats(dh_ctx* ctx, unsigned long long* out);

/* Message describing the last error on the calling thread ("" if none). */
const char* dh_last_error(void);

/* Library version string, e.g. "dh 0.1 sm_100a". */
const char* dh_version(void);

/* ------------------------------------------------------------------------------------------------------------------
 * Periodic multigrid Poisson solver (§6.2 Eqs. 37-48, Appendix C Eqs. C10-C12).
 *
 * Solves A phi = F on the nx x ny x nz torus with cubic cells of size h, A the seven-point Laplacian of Eq. 38
 * (PAPER.md:475).  One cycle = nu1 weighted-Jacobi sweeps (Eq. 39; omega = 2/3), residual (Eq. 41) and
 * 8-cell full-weighting restriction (Eq. 42), gamma recursive visits of the coarse level (1: V-cycle, 2: W-cycle, Eq. C12),
 * trilinear prolongation and correction (Eqs. 44-45), nu2 sweeps.  Levels coarsen by 2 while every extent is even and > 2;
 * the coarsest level gets nu_coarse sweeps (readings A21-A23).
 *
 * Arrays: DEVICE pointers, contiguous [nz][ny][nx] of the context's dtype, 32-byte aligned, owned by the caller, not
 * retained past the call (stream ordered).  The library owns the level hierarchy (about 1.6 extra arrays), allocated in
 * dh_mg_create.  Errors: return code + dh_last_error(); no CPU fallback.  One context per stream, not re-entrant.
 * ------------------------------------------------------------------------------------------------------------------ */
typedef struct dh_mg dh_mg;

enum {
  DH_MG_NU1 = 0,        /* pre-smoothing sweeps, default 2 */
  DH_MG_NU2 = 1,        /* post-smoothing sweeps, default 2 */
  DH_MG_GAMMA = 2,      /* 1 V-cycle (default), 2 W-cycle (the paper's default for gravity) */
  DH_MG_NU_COARSE = 3,  /* Jacobi sweeps on the coarsest level, default 64 */
  DH_MG_OMEGA = 4,      /* Jacobi weight, default 2/3 */
  DH_MG_GRAPH = 5,      /* 1 (default) / 0: replay each cycle as a CUDA graph captured once per (phi, F, options) */
  DH_MG_SUBTREE = 6     /* 1 (default) / 0: a level of <= 4096 cells and every level below it run as ONE kernel (one block, all
                           levels in shared memory) instead of one launch per operator: same operators, same order of operations */
};

dh_mg* dh_mg_create(int nx, int ny, int nz, double h, int dtype);   /* NULL on failure (dh_last_error) */
void dh_mg_destroy(dh_mg* ctx);
int dh_mg_set_stream(dh_mg* ctx, void* cuda_stream);                /* default: legacy stream 0 */
int dh_mg_set_option(dh_mg* ctx, int key, double value);
int dh_mg_levels(const dh_mg* ctx);                                 /* number of grid levels incl. the finest */
long long dh_mg_launches(const dh_mg* ctx);                         /* kernels launched so far (graph nodes counted) */

/* One cycle for A phi = F, in place on phi (in: current iterate, out: next iterate).  F is used as given (it should have
 * zero mean).  Asynchronous on the context's stream. */
int dh_mg_cycle(dh_mg* ctx, void* phi, const void* F);

/* phi = result of `ncycles` cycles from phi = 0 for the zero-mean part of F, mean of phi removed (reading A23).  phi is
 * overwritten, F untouched.  If rel_residual (HOST pointer) is not NULL the call synchronises the stream and stores
 * |F0 - A phi| / |F0| there; otherwise it is asynchronous. */
int dh_mg_solve(dh_mg* ctx, const void* F, void* phi, int ncycles, double* rel_residual);

/* VJP of the converged solve with respect to F (Eqs. 46-48): g_F = A^-1 g_phi, another solve; nothing of
 * the forward solve is stored. */
int dh_mg_solve_vjp(dh_mg* ctx, const void* g_phi, void* g_F, int ncycles, double* rel_residual);

/* ---- Self-gravity as a source term of the hydro step (section 6; the force-class form of PAPER.md:88-107) ----
 * g = -grad phi by second-order central differences on the periodic grid (reading A27), then the operator-split
 * update  u <- u + s_g dt,  s_g = (0, rho g, m . g)  with rho, m of the incoming u.  phi: DEVICE [nz][ny][nx] of the
 * context's dtype (e.g. from dh_mg_solve).  In place, asynchronous on the context's stream; dx_a = L_a / n_a. */
int dh_gravity_source(dh_ctx* ctx, void* U, const void* phi, double dt);

/* Transpose of dh_gravity_source at (U, phi): gU_in = dL/dU (DEVICE state, overwritten), gphi = dL/dphi (DEVICE field,
 * overwritten) from gU_out = dL/d(out).  gU_in must not alias U or gU_out. */
int dh_gravity_source_vjp(dh_ctx* ctx, const void* U, const void* phi, double dt, const void* gU_out, void* gU_in, void* gphi);

/* One self-gravitating step (reading A27): phi from ncycles multigrid cycles on 4 pi G rho of the incoming U (mean removed,
 * reading A23; `mg` must have the grid of `ctx` with h = dx and the same dtype; it is switched to ctx's stream), the hydro step
 * dh_step(U, dt) (cooling, limiter, ... as configured), then the kick dh_gravity_source with that phi.  In place. */
int dh_step_gravity(dh_ctx* ctx, dh_mg* mg, void* U, double dt, double four_pi_g, int ncycles);

/* VJP of dh_step_gravity, dt held constant: through the kick (the post-hydro state is recomputed), the Poisson solve (another
 * solve, Eqs. 46-48) and the hydro step (dh_step_vjp).  U = U^n (pre-step); gU_in overwritten, must not alias U or gU_out. */
int dh_step_gravity_vjp(dh_ctx* ctx, dh_mg* mg, const void* U, double dt, double four_pi_g, int ncycles, const void* gU_out, void* gU_in);

/* ---- Diagnostics (measurements; not part of the path) ----
 * dh_issue_probe times one short instruction mix of the kind the stage kernels consist of (half-rate ALU-pipe FMNMX / LOP3 / FSEL,
 * scalar FADD / FFMA, the packed FADD2 / FMUL2 / FFMA2 of sm_100 in the operand forms the kernels use, alone and combined) on every
 * SM of the current device, with `warps_per_scheduler` (1..4) warps per SM sub-partition and 8 independent chains per thread, and
 * returns the SM cycles (clock64, worst block) per instruction group per scheduler in *cycles_per_group (HOST) and the number of
 * instructions of a group in *instructions_per_group (HOST or NULL).  DESIGN.md section 7b derives the issue bound of
 * stage_fused2_kernel from this table (`python bench.py --issue-probe`; profiles/r02d_issue_bound.md).  Allocates and frees a few
 * KB of device memory and synchronises the device.  mix in [0, DH_ISSUE_PROBE_MIXES); dh_issue_probe_name(mix) is a static string
 * naming the group (NULL for an unknown mix). */
#define DH_ISSUE_PROBE_MIXES 24
int dh_issue_probe(int mix, int warps_per_scheduler, int iters, double* cycles_per_group, int* instructions_per_group);
const char* dh_issue_probe_name(int mix);

#ifdef __cplusplus
}
#endif
#endif /* DH_H_ */
