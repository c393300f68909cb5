// dh_api.cu — the C ABI of include/dh.h: context management, option handling, and the launch sequences of
// dh_cfl_dt / dh_step / dh_step_vjp.  No arithmetic of the scheme lives here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "../../include/dh.h"
#include "dh_internal.cuh"

using namespace dh;

struct dh_ctx : public dh::Ctx {};

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, const char* detail = "") {
  snprintf(g_err, sizeof(g_err), fmt, detail);
  return code;
}
static int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof(g_err), "%s: %s", where, cudaGetErrorString(e));
  return DH_ERR_CUDA;
}
#define DH_CUDA(call, where)                                  \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(e_, where);       \
  } while (0)

namespace dh {
size_t elem_size(const Ctx* c) { return c->dtype == DH_F32 ? 4 : 8; }
void set_error(const char* where, const char* detail) {   // for the other translation units of the library
  if (detail && detail[0]) snprintf(g_err, sizeof(g_err), "%s: %s", where, detail);
  else snprintf(g_err, sizeof(g_err), "%s", where);
}
}  // namespace dh

static size_t state_bytes(const dh_ctx* c) { return 5 * c->N * elem_size(c); }

template <class T>
static Consts<T> make_consts(const dh_ctx* c) {
  Consts<T> k;
  k.gamma = (T)c->gamma;
  k.gm1 = (T)(c->gamma - 1.0);
  k.inv_gm1 = (T)(1.0 / (c->gamma - 1.0));
  k.rho_floor = (T)c->rho_floor;
  k.p_floor = (T)c->p_floor;
  k.lambda0 = (T)c->lambda0;
  k.alpha = (T)c->alpha;
  k.t_floor = (T)c->t_floor;
  k.alpha_is_half = (c->alpha == 0.5);
  k.cool_mode = c->cool_mode;
  k.cool_nsub = c->cool_nsub;
  k.cool_law = (c->cool_law != 0 && c->ntab >= 2) ? 1 : 0;
  k.t_switch = (T)c->t_switch;
  k.lambda1 = (T)c->lambda1; k.alpha1 = (T)c->alpha1; k.lambda2 = (T)c->lambda2; k.alpha2 = (T)c->alpha2;
  k.gamma0 = (T)c->gamma0;
  k.f_sub = (T)c->f_sub;
  k.tab = sizeof(T) == 8 ? (const T*)c->tab_dev_d : (const T*)c->tab_dev;
  k.ntab = c->ntab;
  const double l2_10 = 3.321928094887362;                      // the table is held in log2 units (dh_set_cooling_table)
  k.tab_l2t0 = (T)(c->tab_log10t0 * l2_10);
  k.tab_inv_dl2t = (T)(c->ntab >= 2 ? 1.0 / (c->tab_dlog10t * l2_10) : 0.0);
  return k;
}

static int lazy_alloc(dh_ctx* c, void** slot, size_t bytes, const char* what) {
  if (*slot) return DH_OK;
  cudaError_t e = cudaMalloc(slot, bytes);
  if (e != cudaSuccess) {
    *slot = nullptr;
    cudaGetLastError();
    return fail(DH_ERR_ALLOC, "cudaMalloc failed for %s", what);
  }
  return DH_OK;
}

// Brackets one kernel launch with a pair of events while profiling is on (RAII: start in the constructor,
// stop in the destructor, both on the context's stream).
struct ProfScope {
  dh_ctx* c;
  ProfRec* r;
  ProfScope(dh_ctx* ctx, int kind) : c(ctx), r(nullptr) {
    if (!c->prof_on) return;
    if (c->prof_n == c->prof_cap) {
      int cap = c->prof_cap ? 2 * c->prof_cap : 256;
      ProfRec* q = (ProfRec*)realloc(c->prof, (size_t)cap * sizeof(ProfRec));
      if (!q) return;
      c->prof = q;
      c->prof_cap = cap;
    }
    ProfRec* rec = &c->prof[c->prof_n];
    rec->kind = kind;
    if (cudaEventCreate(&rec->a) != cudaSuccess) return;
    if (cudaEventCreate(&rec->b) != cudaSuccess) { cudaEventDestroy(rec->a); return; }
    cudaEventRecord(rec->a, c->stream);
    c->prof_n += 1;
    r = rec;
  }
  ~ProfScope() {
    if (r) cudaEventRecord(r->b, c->stream);
  }
};

static void prof_drop(dh_ctx* c) {
  for (int i = 0; i < c->prof_n; ++i) { cudaEventDestroy(c->prof[i].a); cudaEventDestroy(c->prof[i].b); }
  c->prof_n = 0;
}

// A context lives on the device that was current at dh_create (its scratch, its kernels' attributes): calling it with
// another device current would launch there on foreign pointers.
static int check_device(const dh_ctx* c, const char* who) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) {
    snprintf(g_err, sizeof(g_err), "%s: the context belongs to device %d but device %d is current (cudaSetDevice first)", who, c->device, dev);
    return DH_ERR_ARG;
  }
  return DH_OK;
}

extern "C" {

const char* dh_last_error(void) { return g_err; }
const char* dh_version(void) { return "dh 0.1 sm_100a"; }

dh_ctx* dh_create(int nx, int ny, int nz, double gamma, int dtype) {
  g_err[0] = 0;
  if (nx < 4 || ny < 4 || nz < 4) { fail(DH_ERR_ARG, "dh_create: every n_a must be >= 4%s"); return nullptr; }
  if (!(gamma > 1.0) || !isfinite(gamma)) { fail(DH_ERR_ARG, "dh_create: gamma must be finite and > 1%s"); return nullptr; }
  if (dtype != DH_F32 && dtype != DH_F64) { fail(DH_ERR_ARG, "dh_create: dtype must be DH_F32 or DH_F64%s"); return nullptr; }
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cuda_fail(e, "dh_create: cudaGetDevice (no CUDA device? there is no CPU fallback)"); return nullptr; }
  dh_ctx* c = new (std::nothrow) dh_ctx();
  if (!c) { fail(DH_ERR_ALLOC, "dh_create: out of host memory%s"); return nullptr; }
  memset(static_cast<dh::Ctx*>(c), 0, sizeof(dh::Ctx));
  c->nx = nx; c->ny = ny; c->nz = nz; c->dtype = dtype;
  c->N = (size_t)nx * ny * nz;
  c->gamma = gamma;
  c->cfl = 0.4;
  c->L[0] = c->L[1] = c->L[2] = 1.0;
  c->cooling = 0; c->kernel = 0; c->limiter = 0; c->riemann = 0; c->integrator = 0; c->cool_mode = 0; c->cool_nsub = 1; c->fuse_cfl = 1; c->c_cool = 0.0; c->dt_max = 0.0;
  c->lambda0 = 1e-3; c->alpha = 0.5; c->t_floor = 0.01;
  c->cool_law = 0; c->t_switch = 1.0; c->lambda1 = 0.0; c->alpha1 = 1.0; c->lambda2 = 0.0; c->alpha2 = 0.5; c->gamma0 = 0.0; c->f_sub = 0.1;
  c->ntab = 0; c->tab_log10t0 = 0.0; c->tab_dlog10t = 1.0;
  c->rho_floor = 1e-10; c->p_floor = 1e-10;
  c->stream = 0;
  c->device = dev;
  cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (c->sm_count <= 0) c->sm_count = 148;
  bool ok = cudaMalloc(&c->Us, state_bytes(c)) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&c->acc, 8 * sizeof(unsigned long long)) == cudaSuccess;
  ok = ok && cudaMalloc(&c->dt_dev, 8) == cudaSuccess;
  ok = ok && cudaMalloc((void**)&c->result_dev, sizeof(CflResult)) == cudaSuccess;
  ok = ok && cudaMallocHost((void**)&c->result_host, sizeof(CflResult)) == cudaSuccess;
  ok = ok && cudaMemset(c->acc, 0, 8 * sizeof(unsigned long long)) == cudaSuccess;
  {
    const unsigned long long inf_bits = 0x7ff0000000000000ull;   // slot [4]: running min of t_cool (Eq. 20), armed with +inf
    ok = ok && cudaMemcpy(c->acc + 4, &inf_bits, sizeof(inf_bits), cudaMemcpyHostToDevice) == cudaSuccess;
  }
  ok = ok && cudaMemset(c->dt_dev, 0, 8) == cudaSuccess;
  ok = ok && cudaMemset(c->result_dev, 0, sizeof(CflResult)) == cudaSuccess;
  if (!ok) {
    cudaError_t le = cudaGetLastError();
    dh_destroy(c);
    snprintf(g_err, sizeof(g_err), "dh_create: allocation failed (%s)", cudaGetErrorString(le));
    return nullptr;
  }
  memset(c->result_host, 0, sizeof(CflResult));
  return c;
}

void dh_destroy(dh_ctx* c) {
  if (!c) return;
  void* dev[] = {c->Us, c->gs, c->Ub, c->Uc, c->ga, c->cand_list, c->cand_cnt, c->cand_thr, c->cand_stats, c->U1, c->g1, c->Uhost_dev, c->Uhost_dev2, c->gA, c->gB, c->rev_scratch, c->adj_states, c->adj_dts_dev, c->acc, c->dt_dev, c->result_dev, c->tab_dev, c->tab_dev_d, c->tab_part, c->grav_phi, c->grav_F, c->grav_gb, c->grav_U1, c->grav_g1};
  for (void* p : dev)
    if (p) cudaFree(p);
  if (c->result_host) cudaFreeHost(c->result_host);
  if (c->adj_dts_host) cudaFreeHost(c->adj_dts_host);
  for (int i = 0; i < 3 * c->ev_n; ++i) cudaEventDestroy(c->ev_slab[i]);
  free(c->ev_slab);
  if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
  if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
  prof_drop(c);
  free(c->prof);
  delete c;
}

int dh_set_stream(dh_ctx* c, void* cuda_stream) {
  if (!c) return fail(DH_ERR_ARG, "dh_set_stream: NULL context%s");
  c->stream = (cudaStream_t)cuda_stream;
  return DH_OK;
}

int dh_set_option(dh_ctx* c, int key, double v) {
  if (!c) return fail(DH_ERR_ARG, "dh_set_option: NULL context%s");
  if (!isfinite(v)) return fail(DH_ERR_ARG, "dh_set_option: value must be finite%s");
  switch (key) {
    case DH_OPT_CFL: if (v <= 0) return fail(DH_ERR_ARG, "dh_set_option: CFL must be > 0%s"); c->cfl = v; break;
    case DH_OPT_LX: case DH_OPT_LY: case DH_OPT_LZ:
      if (v <= 0) return fail(DH_ERR_ARG, "dh_set_option: box length must be > 0%s");
      c->L[key - DH_OPT_LX] = v; break;
    case DH_OPT_COOLING: c->cooling = (v != 0.0); break;
    case DH_OPT_LAMBDA0: if (v < 0) return fail(DH_ERR_ARG, "dh_set_option: lambda0 must be >= 0%s"); c->lambda0 = v; break;
    case DH_OPT_ALPHA: c->alpha = v; break;   /* any finite exponent; the rate is 0 for T <= 0 whatever alpha (cool_rate) */
    case DH_OPT_T_FLOOR: if (v < 0) return fail(DH_ERR_ARG, "dh_set_option: t_floor must be >= 0%s"); c->t_floor = v; break;
    case DH_OPT_RHO_FLOOR: if (v <= 0) return fail(DH_ERR_ARG, "dh_set_option: floors must be > 0%s"); c->rho_floor = v; break;
    case DH_OPT_P_FLOOR: if (v <= 0) return fail(DH_ERR_ARG, "dh_set_option: floors must be > 0%s"); c->p_floor = v; break;
    case DH_OPT_KERNEL: if (v != 0.0 && v != 1.0) return fail(DH_ERR_ARG, "dh_set_option: kernel must be 0 or 1%s"); c->kernel = (int)v; break;
    case DH_OPT_REV_SLAB: if (v < 0 || v != (double)(int)v) return fail(DH_ERR_ARG, "dh_set_option: rev_slab must be a non-negative integer%s"); c->rev_slab_opt = (int)v; break;
    case DH_OPT_LIMITER: if (v != 0.0 && v != 1.0 && v != 2.0) return fail(DH_ERR_ARG, "dh_set_option: limiter must be 0, 1 or 2%s"); c->limiter = (int)v; break;
    case DH_OPT_INTEGRATOR: if (v != 0.0 && v != 1.0 && v != 2.0) return fail(DH_ERR_ARG, "dh_set_option: integrator must be 0, 1 or 2%s"); c->integrator = (int)v; break;
    case DH_OPT_FUSE_CFL: c->fuse_cfl = (v != 0.0); break;
    case DH_OPT_C_COOL: if (!(v >= 0.0) || !isfinite(v)) return fail(DH_ERR_ARG, "dh_set_option: c_cool must be finite and >= 0%s"); c->c_cool = v; break;
    case DH_OPT_DT_MAX: if (!(v >= 0.0) || !isfinite(v)) return fail(DH_ERR_ARG, "dh_set_option: dt_max must be finite and >= 0%s"); c->dt_max = v; break;
    case DH_OPT_RIEMANN: if (v != 0.0 && v != 1.0 && v != 2.0) return fail(DH_ERR_ARG, "dh_set_option: riemann must be 0, 1 or 2%s"); c->riemann = (int)v; break;
    case DH_OPT_COOL_MODE: if (v != 0.0 && v != 1.0 && v != 2.0) return fail(DH_ERR_ARG, "dh_set_option: cool_mode must be 0, 1 or 2%s"); c->cool_mode = (int)v; break;
    case DH_OPT_COOL_LAW:
      if (v != 0.0 && v != 1.0) return fail(DH_ERR_ARG, "dh_set_option: cool_law must be 0 or 1%s");
      if (v == 1.0 && c->ntab < 2) return fail(DH_ERR_ARG, "dh_set_option: cool_law = 1 needs a table (dh_set_cooling_table first)%s");
      c->cool_law = (int)v; break;
    case DH_OPT_T_SWITCH: if (!(v > 0)) return fail(DH_ERR_ARG, "dh_set_option: t_switch must be > 0%s"); c->t_switch = v; break;
    case DH_OPT_LAMBDA1: if (v < 0) return fail(DH_ERR_ARG, "dh_set_option: lambda1 must be >= 0%s"); c->lambda1 = v; break;
    case DH_OPT_ALPHA1: c->alpha1 = v; break;
    case DH_OPT_LAMBDA2: if (v < 0) return fail(DH_ERR_ARG, "dh_set_option: lambda2 must be >= 0%s"); c->lambda2 = v; break;
    case DH_OPT_ALPHA2: c->alpha2 = v; break;
    case DH_OPT_GAMMA0: if (v < 0) return fail(DH_ERR_ARG, "dh_set_option: gamma0 must be >= 0%s"); c->gamma0 = v; break;
    case DH_OPT_COOL_FSUB: if (!(v > 0)) return fail(DH_ERR_ARG, "dh_set_option: cool_fsub must be > 0%s"); c->f_sub = v; break;
    case DH_OPT_STREAM_SLAB: if (v < 0 || v != (double)(int)v) return fail(DH_ERR_ARG, "dh_set_option: stream_slab must be a non-negative integer%s"); c->stream_slab_opt = (int)v; break;
    case DH_OPT_COOL_NSUB:
      if (v < 1 || v > DH_COOL_NSUB_MAX || v != (double)(int)v) return fail(DH_ERR_ARG, "dh_set_option: cool_nsub must be an integer in 1 .. 64%s");
      c->cool_nsub = (int)v; break;
    default: return fail(DH_ERR_ARG, "dh_set_option: unknown key%s");
  }
  return DH_OK;
}

int dh_get_option(const dh_ctx* c, int key, double* out) {
  if (!c || !out) return fail(DH_ERR_ARG, "dh_get_option: NULL argument%s");
  switch (key) {
    case DH_OPT_CFL: *out = c->cfl; break;
    case DH_OPT_LX: case DH_OPT_LY: case DH_OPT_LZ: *out = c->L[key - DH_OPT_LX]; break;
    case DH_OPT_COOLING: *out = c->cooling; break;
    case DH_OPT_LAMBDA0: *out = c->lambda0; break;
    case DH_OPT_ALPHA: *out = c->alpha; break;
    case DH_OPT_T_FLOOR: *out = c->t_floor; break;
    case DH_OPT_RHO_FLOOR: *out = c->rho_floor; break;
    case DH_OPT_P_FLOOR: *out = c->p_floor; break;
    case DH_OPT_KERNEL: *out = c->kernel; break;
    case DH_OPT_LIMITER: *out = c->limiter; break;
    case DH_OPT_REV_SLAB: *out = c->rev_slab_opt; break;
    case DH_OPT_INTEGRATOR: *out = c->integrator; break;
    case DH_OPT_FUSE_CFL: *out = c->fuse_cfl; break;
    case DH_OPT_C_COOL: *out = c->c_cool; break;
    case DH_OPT_DT_MAX: *out = c->dt_max; break;
    case DH_OPT_RIEMANN: *out = c->riemann; break;
    case DH_OPT_COOL_MODE: *out = c->cool_mode; break;
    case DH_OPT_COOL_LAW: *out = c->cool_law; break;
    case DH_OPT_T_SWITCH: *out = c->t_switch; break;
    case DH_OPT_LAMBDA1: *out = c->lambda1; break;
    case DH_OPT_ALPHA1: *out = c->alpha1; break;
    case DH_OPT_LAMBDA2: *out = c->lambda2; break;
    case DH_OPT_ALPHA2: *out = c->alpha2; break;
    case DH_OPT_GAMMA0: *out = c->gamma0; break;
    case DH_OPT_COOL_FSUB: *out = c->f_sub; break;
    case DH_OPT_STREAM_SLAB: *out = c->stream_slab_opt; break;
    case DH_OPT_COOL_NSUB: *out = c->cool_nsub; break;
    default: return fail(DH_ERR_ARG, "dh_get_option: unknown key%s");
  }
  return DH_OK;
}

unsigned long long dh_launch_count(const dh_ctx* c) { return c ? c->launches : 0ull; }

int dh_profile_enable(dh_ctx* c, int on) {
  if (!c) return fail(DH_ERR_ARG, "dh_profile_enable: NULL context%s");
  if (!on) {
    DH_CUDA(cudaStreamSynchronize(c->stream), "dh_profile_enable: synchronize");
    prof_drop(c);
  }
  c->prof_on = on ? 1 : 0;
  return DH_OK;
}

int dh_profile_read(dh_ctx* c, double* ms_out, unsigned long long* launches_out) {
  if (!c) return fail(DH_ERR_ARG, "dh_profile_read: NULL context%s");
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_profile_read: synchronize");
  for (int i = 0; i < c->prof_n; ++i) {
    const ProfRec& r = c->prof[i];
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess && r.kind >= 0 && r.kind < DH_K_COUNT_) {
      if (ms_out) ms_out[r.kind] += (double)ms;
      if (launches_out) launches_out[r.kind] += 1ull;
    }
  }
  prof_drop(c);
  return DH_OK;
}

}  // extern "C"

// dh_advance / dh_stream_host: the CFL candidate list of DH_OPT_FUSE_CFL, allocated on first use, counters reset per call
static int cand_alloc(dh_ctx* c) {
  if (!c->cand_list) {
    c->cand_cap = 1u << 20;
    int rc = lazy_alloc(c, (void**)&c->cand_list, (size_t)c->cand_cap * sizeof(unsigned), "the CFL candidate list");
    if (rc) return rc;
    rc = lazy_alloc(c, (void**)&c->cand_cnt, 2 * sizeof(unsigned), "the CFL candidate counters");
    if (rc) return rc;
    rc = lazy_alloc(c, &c->cand_thr, 16, "the CFL candidate thresholds");
    if (rc) return rc;
    rc = lazy_alloc(c, (void**)&c->cand_stats, 3 * sizeof(unsigned long long), "the CFL candidate counters");
    if (rc) return rc;
    DH_CUDA(cudaMemsetAsync(c->cand_stats, 0, 3 * sizeof(unsigned long long), c->stream), "reset of the candidate statistics");
  }
  DH_CUDA(cudaMemsetAsync(c->cand_cnt, 0, 2 * sizeof(unsigned), c->stream), "reset of the candidate counters");
  return DH_OK;
}

// ------------------------------------------------------------------------------------------------ CFL
// cand: the state was written by a last stage that pushed its CFL candidates (dh_advance): exact recipe on those
// packs, then the full reduction only if they do not settle the maxima
template <class T>
static int cfl_launch(dh_ctx* c, const void* U, bool cand = false, bool force_tcool = false) {
  CflParams<T> p;
  // Eq. 21: the reduction also evaluates Eq. 20 when cooling is on and c_cool > 0 (or for dh_cool_tmin)
  p.cool_lim = (force_tcool || (c->cooling != 0 && c->c_cool > 0.0)) ? 1 : 0;
  p.gm1d = c->gamma - 1.0; p.lambda0 = c->lambda0; p.alpha = c->alpha; p.c_cool = c->cooling != 0 ? c->c_cool : 0.0; p.dt_max = c->dt_max;
  p.cd = make_consts<double>(c);                    // Eq. 20 with the law of DH_OPT_COOL_LAW, in double
  if (p.cool_lim) cand = false;
  p.U = (const T*)U;
  p.N = c->N;
  p.gamma = (T)c->gamma;
  p.gm1 = (T)(c->gamma - 1.0);
  p.rho_floor = (T)c->rho_floor;
  p.p_floor = (T)c->p_floor;
  const int n[3] = {c->nx, c->ny, c->nz};
  for (int a = 0; a < 3; ++a) p.dx[a] = (T)(c->L[a] / n[a]);
  p.cfl = (T)c->cfl;
  p.acc = c->acc;
  p.dt_dev = (T*)c->dt_dev;
  p.result = c->result_dev;
  p.cand_list = c->cand_list; p.cand_cnt = c->cand_cnt; p.cand_thr = (T*)c->cand_thr; p.cand_cap = c->cand_cap; p.cand_stats = c->cand_stats;
  {
    ProfScope ps(c, cand ? DH_K_CFL_CAND : DH_K_CFL_REDUCE);
    if (cand) {
      DH_CUDA(launch_cfl_candidates<T>(p, c->sm_count, c->stream), "dh_advance: CFL candidate kernel launch");
      c->launches += 2;
    } else {
      DH_CUDA(launch_cfl_reduce<T>(p, c->sm_count, c->stream), "dh_cfl_dt: reduction kernel launch");
      c->launches += 1;
    }
  }
  {
    ProfScope ps(c, DH_K_CFL_FINISH);
    DH_CUDA(launch_cfl_finish<T>(p, c->stream), "dh_cfl_dt: epilogue kernel launch");
  }
  c->launches += 1;
  return DH_OK;
}

// ------------------------------------------------------------------------------------------ forward
// What only the fused kernel can do: a z range of planes (dh_stream_host) and the base state formed in the kernel as
// wB B + wX U (the Shu-Osher stages of Heun / SSPRK3)
struct StageExtra {
  int zbeg = 0, zcnt = 0;
  bool combo = false;
  double wB = 1.0, wX = 0.0;
};
static bool fused_ok(const dh_ctx* c) { return c->kernel == 0 && c->nx % 2 == 0 && (c->ny + 5) / 6 <= 65535; }
// the in-kernel combination is compiled for fp64 and for the fp32 kernel with 16-byte staging copies (nx % 4 == 0)
static bool combo_ok(const dh_ctx* c) { return fused_ok(c) && (c->dtype == DH_F64 || c->nx % 4 == 0); }

template <class T>
static int stage_launch(dh_ctx* c, int kind, const void* U, const void* B, void* out, double dt, bool devdt, double frac, bool cool,
                        bool cand = false, const StageExtra& x = StageExtra()) {
  if ((x.zcnt != 0 && !fused_ok(c)) || (x.combo && !combo_ok(c))) return fail(DH_ERR_ARG, "stage_launch: z ranges and in-kernel combinations need the fused kernel%s");
  StageParams<T> p;
  p.zbeg = x.zbeg; p.zcnt = x.zcnt ? x.zcnt : c->nz;
  p.combo = x.combo ? 1 : 0; p.wB = (T)x.wB; p.wX = (T)x.wX;
  p.U = (const T*)U; p.B = (const T*)B; p.out = (T*)out;
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
  const int n[3] = {c->nx, c->ny, c->nz};
  for (int a = 0; a < 3; ++a) p.inv_dx[a] = (T)(n[a] / c->L[a]);
  p.dt = (T)dt;
  p.dt_dev = devdt ? (const T*)c->dt_dev : nullptr;
  p.frac = (T)frac;
  p.cool = cool ? 1 : 0;
  p.c = make_consts<T>(c);
  p.cand_list = nullptr; p.cand_cnt = nullptr; p.cand_thr = nullptr; p.cand_cap = 0;
  if (cand && c->kernel == 0 && c->cand_list && c->N < ((size_t)1 << 32)) {
    p.cand_list = c->cand_list; p.cand_cnt = c->cand_cnt; p.cand_thr = (const T*)c->cand_thr; p.cand_cap = c->cand_cap;
  }
  c->cand_ok = 0;
  ProfScope ps(c, kind);
  bool done = false;
  if (c->kernel == 0) {
    bool supported = false;
    cudaError_t e = launch_stage_fused2<T>(p, c->limiter, c->riemann, c->sm_count, c->stream, &supported);
    if (supported) {
      if (e != cudaSuccess) return cuda_fail(e, "dh_step: fused stage kernel launch");
      done = true;
      c->cand_ok = p.cand_list != nullptr;      // only this kernel pushes candidates
    }
  }
  if (!done) DH_CUDA(launch_stage_naive<T>(p, c->limiter, c->riemann, c->stream), "dh_step: stage kernel launch");
  c->launches += 1;
  return DH_OK;
}

// out = a X + b Y over a whole state (Y may be NULL); the base states and scaled cotangents of Heun / SSPRK3
template <class T>
static int lincomb(dh_ctx* c, void* out, double a, const void* X, double b, const void* Y) {
  ProfScope ps(c, DH_K_LINCOMB);
  DH_CUDA(launch_lincomb<T>((T*)out, (T)a, (const T*)X, (T)b, (const T*)Y, 5 * c->N, c->sm_count, c->stream), "lincomb kernel launch");
  c->launches += 1;
  return DH_OK;
}

// The stage states of Heun / SSPRK3 up to (not including) the last stage: c->Us = U1, (SSPRK3) c->Uc = U2, and
// c->Ub = the base state of the last stage.  *last_in = the state the last stage differentiates, *last_frac its weight.
template <class T>
static int rk_prefix(dh_ctx* c, const void* U, double dt, bool devdt, const void** last_in, double* last_frac) {
  int rc = lazy_alloc(c, &c->Ub, state_bytes(c), "the base-state combination");
  if (rc) return rc;
  rc = stage_launch<T>(c, DH_K_STAGE1, U, U, c->Us, dt, devdt, 1.0, false);              // U1 = U - dt D(U)
  if (rc) return rc;
  if (combo_ok(c)) {
    // the combinations are formed inside the stage kernel (StageExtra::combo); *last_in / *last_frac as below, rk_last()
    // passes the weights of the last stage itself
    if (c->integrator == 1) { *last_in = c->Us; *last_frac = 0.5; return DH_OK; }
    rc = lazy_alloc(c, &c->Uc, state_bytes(c), "the second stage state");
    if (rc) return rc;
    StageExtra x;
    x.combo = true; x.wB = 0.75; x.wX = 0.25;
    rc = stage_launch<T>(c, DH_K_STAGE1, c->Us, U, c->Uc, dt, devdt, 0.25, false, false, x);   // U2 = 3/4 U + 1/4 U1 - 1/4 dt D(U1)
    *last_in = c->Uc; *last_frac = 2.0 / 3.0;
    return rc;
  }
  if (c->integrator == 1) {                                                                // Heun
    rc = lincomb<T>(c, c->Ub, 0.5, U, 0.5, c->Us);
    *last_in = c->Us; *last_frac = 0.5;
    return rc;
  }
  rc = lazy_alloc(c, &c->Uc, state_bytes(c), "the second stage state");
  if (rc) return rc;
  rc = lincomb<T>(c, c->Ub, 0.75, U, 0.25, c->Us);
  if (rc) return rc;
  rc = stage_launch<T>(c, DH_K_STAGE1, c->Us, c->Ub, c->Uc, dt, devdt, 0.25, false);      // U2 = 3/4 U + 1/4 (U1 - dt D(U1))
  if (rc) return rc;
  rc = lincomb<T>(c, c->Ub, 1.0 / 3.0, U, 2.0 / 3.0, c->Uc);
  *last_in = c->Uc; *last_frac = 2.0 / 3.0;
  return rc;
}

// The last stage of Heun / SSPRK3 after rk_prefix:  out = (1 - w) U + w (X - dt D(X)),  X = last_in
template <class T>
static int rk_last(dh_ctx* c, const void* last_in, double w, const void* U, void* out, double dt, bool devdt, bool cool, bool cand) {
  if (!combo_ok(c)) return stage_launch<T>(c, DH_K_STAGE2, last_in, c->Ub, out, dt, devdt, w, cool, cand);
  StageExtra x;
  x.combo = true; x.wB = c->integrator == 1 ? 0.5 : 1.0 / 3.0; x.wX = w;
  return stage_launch<T>(c, DH_K_STAGE2, last_in, U, out, dt, devdt, w, cool, cand, x);
}

// The cooling integrators the stage kernels do not fuse (sub-cycled Eq. 23 with N_sub > 1, trapezoid Eq. 22): one
// streaming pass over the finished state (reads 5 words per cell, rewrites E).
template <class T>
static int cool_launch(dh_ctx* c, void* U, double dt, bool devdt) {
  ProfScope ps(c, DH_K_COOL);
  DH_CUDA(launch_cool_fwd<T>((T*)U, c->N, (T)dt, devdt ? (const T*)c->dt_dev : nullptr, make_consts<T>(c), c->stream),
          "dh_step: cooling kernel launch");
  c->launches += 1;
  return DH_OK;
}

template <class T>
static int step_impl(dh_ctx* c, void* U, double dt, bool devdt, bool cand = false) {
  // default cooling update (Eq. 23, N_sub = 1): epilogue of the last stage; the others: a pass of their own, and the
  // CFL candidates (pushed by the last stage from the pre-cooling values) are not used
  const bool split_cool = c->cooling != 0 && (c->cool_mode != 0 || c->cool_nsub > 1 || c->cool_law != 0);
  const bool fused_cool = c->cooling != 0 && !split_cool;
  if (c->integrator != 0) {
    // Heun / SSPRK3 in Shu-Osher form: every stage is  out = B - w dt D(state)
    const void* last_in = nullptr;
    double w = 0.0;
    int rc = rk_prefix<T>(c, U, dt, devdt, &last_in, &w);
    if (rc) return rc;
    rc = rk_last<T>(c, last_in, w, U, U, dt, devdt, fused_cool, cand && !split_cool);
    if (rc || !split_cool) return rc;
    return cool_launch<T>(c, U, dt, devdt);
  }
  // predictor: U* = U^n - dt/2 D(U^n)   (Eq. A6);  corrector, in place: U^{n+1} = U^n - dt D(U*)   (Eq. A7)
  int rc = stage_launch<T>(c, DH_K_STAGE1, U, U, c->Us, dt, devdt, 0.5, false);
  if (rc) return rc;
  rc = stage_launch<T>(c, DH_K_STAGE2, c->Us, U, U, dt, devdt, 1.0, fused_cool, cand && !split_cool);
  if (rc || !split_cool) return rc;
  return cool_launch<T>(c, U, dt, devdt);
}

// ------------------------------------------------------------------------------------------ reverse
template <class T>
static int rev_launch(dh_ctx* c, int kind, const void* U, const void* g, const void* b1, const void* b2, void* out, double dt, double frac,
                      double w1, double w2) {
  RevParams<T> p;
  p.U = (const T*)U; p.g = (const T*)g; p.b1 = (const T*)b1; p.b2 = (const T*)b2; p.out = (T*)out;
  p.w1 = (T)w1; p.w2 = (T)w2;
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
  const int n[3] = {c->nx, c->ny, c->nz};
  for (int a = 0; a < 3; ++a) p.inv_dx[a] = (T)(n[a] / c->L[a]);
  p.dt = (T)dt;
  p.frac = (T)frac;
  p.c = make_consts<T>(c);
  ProfScope ps(c, kind);
  DH_CUDA(launch_rev_naive<T>(p, c->limiter, c->riemann, c->stream), "dh_step_vjp: reverse stage kernel launch");
  c->launches += 1;
  return DH_OK;
}

// Fused reversed stage (dh_rev.cu): per z slab, the face-adjoint sweep over the slab (it reads 3 planes on each side), then
// the gather over the slab.  The scratch (10 words per cell of a slab + the tile-edge array) is allocated on first use.
template <class T>
static int rev_fused(dh_ctx* c, int kind, const void* U, const void* g, const void* b1, const void* b2, void* out, double dt, double frac,
                     double w1, double w2) {
  const size_t NP = (size_t)c->nx * c->ny;
  const int ntx = (c->nx + 63) / 64;                       // tiles per row of rev_faces_kernel (RTX = 64)
  const size_t EP = (size_t)c->ny * ntx * 2;               // tile-edge words per plane and field
  const int want = c->rev_slab_opt > 0 ? (c->rev_slab_opt < c->nz ? c->rev_slab_opt : c->nz) : 0;
  const int words = rev_scratch_words(c->limiter);
  if (c->rev_scratch && ((want > 0 && want != c->rev_slab) || words != c->rev_words)) {      // an option changed: resize
    DH_CUDA(cudaStreamSynchronize(c->stream), "dh_step_vjp: synchronize");
    cudaFree(c->rev_scratch);
    c->rev_scratch = nullptr;
  }
  if (!c->rev_scratch) {
    const size_t per_plane = ((size_t)words * NP + 5 * EP) * elem_size(c);
    long long planes = want;
    if (planes == 0) {
      size_t free_b = 0, total_b = 0;
      if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); free_b = (size_t)8 << 30; }
      size_t budget = (size_t)48 << 30;                    // one slab at 1024^3 fp32 (43 GB) when the memory is there
      if (budget > free_b / 10 * 7) budget = free_b / 10 * 7;
      planes = (long long)(budget / per_plane);
      if (planes > c->nz) planes = c->nz;
    }
    if (planes < 1) return fail(DH_ERR_ALLOC, "dh_step_vjp: not enough device memory for the reverse-stage scratch%s");
    int rc = lazy_alloc(c, &c->rev_scratch, (size_t)planes * per_plane, "the reverse-stage scratch");
    if (rc) return rc;
    c->rev_slab = (int)planes;
    c->rev_words = words;
  }
  const int SP = c->rev_slab;
  const int n[3] = {c->nx, c->ny, c->nz};
  RevFaceParams<T> a;
  a.U = (const T*)U; a.g = (const T*)g;
  a.Wp = (T*)c->rev_scratch;
  a.C = a.Wp + (size_t)5 * SP * NP;
  a.Ce = a.C + (size_t)(words - 5) * SP * NP;
  a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
  a.sp0 = 0; a.SP = SP; a.ntx = ntx; a.SPE = (size_t)SP * EP;
  for (int k = 0; k < 3; ++k) a.coef[k] = (T)(frac * dt * n[k] / c->L[k]);
  a.c = make_consts<T>(c);
  RevGatherParams<T> b;
  b.U = (const T*)U; b.Wp = a.Wp; b.C = a.C; b.Ce = a.Ce; b.b1 = (const T*)b1; b.b2 = (const T*)b2; b.out = (T*)out;
  b.w1 = (T)w1; b.w2 = (T)w2;
  b.nx = c->nx; b.ny = c->ny; b.nz = c->nz; b.sp0 = 0; b.SP = SP; b.ntx = ntx; b.SPE = a.SPE; b.c = a.c;
  ProfScope ps(c, kind);
  for (int z0 = 0; z0 < c->nz; z0 += c->rev_slab) {
    const int nplanes = (c->nz - z0 < c->rev_slab) ? c->nz - z0 : c->rev_slab;
    a.zs = z0; a.nout = nplanes;
    DH_CUDA(launch_rev_faces<T>(a, c->limiter, c->riemann, c->sm_count, c->stream), "dh_step_vjp: face-adjoint kernel launch");
    b.z0 = z0; b.nplanes = nplanes;
    DH_CUDA(launch_rev_gather<T>(b, c->limiter, c->stream), "dh_step_vjp: gather kernel launch");
    c->launches += 2;
  }
  return DH_OK;
}

template <class T>
static int rev_stage(dh_ctx* c, int kind, const void* U, const void* g, const void* b1, const void* b2, void* out, double dt, double frac,
                     double w1 = 1.0, double w2 = 1.0) {
  // the fused pair handles every limiter and Riemann flux on even nx; odd nx and DH_OPT_KERNEL = 1 take the one-thread-per-cell gather kernel
  if (c->kernel == 0 && c->nx % 2 == 0) return rev_fused<T>(c, kind, U, g, b1, b2, out, dt, frac, w1, w2);
  return rev_launch<T>(c, kind, U, g, b1, b2, out, dt, frac, w1, w2);
}

// VJP of a Heun / SSPRK3 step.  With a = w g (w the last stage's weight) the last stage gives
// Xbar = a - dt J_D(X)^T a for its input X, and so on down to U; the U-weights of the base states add w_U g terms.
template <class T>
static int vjp_rk(dh_ctx* c, const void* U, double dt, const void* gout, void* gin) {
  int rc = lazy_alloc(c, &c->gs, state_bytes(c), "the stage cotangent");
  if (rc) return rc;
  const void* last_in = nullptr;
  double w = 0.0;
  rc = rk_prefix<T>(c, U, dt, false, &last_in, &w);                // recompute the stage states (nothing was stored)
  if (rc) return rc;
  const void* g1 = gout;
  if (c->cooling) {
    rc = lazy_alloc(c, &c->U1, state_bytes(c), "the pre-cooling state");
    if (rc) return rc;
    rc = lazy_alloc(c, &c->g1, state_bytes(c), "the pre-cooling cotangent");
    if (rc) return rc;
    rc = rk_last<T>(c, last_in, w, U, c->U1, dt, false, false, false);
    if (rc) return rc;
    ProfScope ps(c, DH_K_COOL_VJP);
    DH_CUDA(launch_cool_vjp<T>((const T*)c->U1, (const T*)gout, (T*)c->g1, c->N, (T)dt, make_consts<T>(c), c->stream),
            "dh_step_vjp: cooling reverse kernel launch");
    c->launches += 1;
    g1 = c->g1;
  }
  void* const h = c->Ub;                                           // the base state is dead: a combined cotangent lives there
  if (c->integrator == 1) {
    // Heun: U' = 1/2 U + 1/2 (U1 - dt D(U1)), U1 = U - dt D(U)
    rc = rev_stage<T>(c, DH_K_REV2, c->Us, g1, g1, nullptr, c->gs, dt, 0.5, 0.5);    // U1bar = 1/2 g1 - dt/2 J_D(U1)^T g1
    if (rc) return rc;
    return rev_stage<T>(c, DH_K_REV1, U, c->gs, g1, c->gs, gin, dt, 1.0, 0.5, 1.0);  // Ubar = 1/2 g1 + U1bar - dt J_D(U)^T U1bar
  }
  // SSPRK3: U' = 1/3 U + 2/3 (U2 - dt D(U2)), U2 = 3/4 U + 1/4 (U1 - dt D(U1)), U1 = U - dt D(U)
  rc = lazy_alloc(c, &c->ga, state_bytes(c), "the first stage cotangent");
  if (rc) return rc;
  rc = rev_stage<T>(c, DH_K_REV2, c->Uc, g1, g1, nullptr, c->gs, dt, 2.0 / 3.0, 2.0 / 3.0);   // U2bar = 2/3 g1 - 2/3 dt J_D(U2)^T g1
  if (rc) return rc;
  rc = rev_stage<T>(c, DH_K_REV1, c->Us, c->gs, c->gs, nullptr, c->ga, dt, 0.25, 0.25);       // U1bar = 1/4 U2bar - 1/4 dt J_D(U1)^T U2bar
  if (rc) return rc;
  rc = lincomb<T>(c, h, 1.0 / 3.0, g1, 0.75, c->gs);
  if (rc) return rc;
  return rev_stage<T>(c, DH_K_REV1, U, c->ga, h, c->ga, gin, dt, 1.0);               // Ubar = 1/3 g1 + 3/4 U2bar + U1bar - dt J_D(U)^T U1bar
}

template <class T>
static int vjp_impl(dh_ctx* c, const void* U, double dt, const void* gout, void* gin) {
  if (c->integrator != 0) return vjp_rk<T>(c, U, dt, gout, gin);
  int rc = lazy_alloc(c, &c->gs, state_bytes(c), "the U* cotangent state");
  if (rc) return rc;
  // recompute U* = U^n - dt/2 D(U^n)  (nothing was stored by dh_step)
  rc = stage_launch<T>(c, DH_K_STAGE1, U, U, c->Us, dt, false, 0.5, false);
  if (rc) return rc;
  const void* g1 = gout;
  if (c->cooling) {
    // pre-cooling state U1 = U^n - dt D(U*), then g1 = J_cool(U1)^T g_out
    rc = lazy_alloc(c, &c->U1, state_bytes(c), "the pre-cooling state");
    if (rc) return rc;
    rc = lazy_alloc(c, &c->g1, state_bytes(c), "the pre-cooling cotangent");
    if (rc) return rc;
    rc = stage_launch<T>(c, DH_K_STAGE2, c->Us, U, c->U1, dt, false, 1.0, false);
    if (rc) return rc;
    ProfScope ps(c, DH_K_COOL_VJP);
    DH_CUDA(launch_cool_vjp<T>((const T*)c->U1, (const T*)gout, (T*)c->g1, c->N, (T)dt, make_consts<T>(c), c->stream),
            "dh_step_vjp: cooling reverse kernel launch");
    c->launches += 1;
    g1 = c->g1;
  }
  // reverse corrector:  gs = -dt J_D(U*)^T g1
  rc = rev_stage<T>(c, DH_K_REV2, c->Us, g1, nullptr, nullptr, c->gs, dt, 1.0);
  if (rc) return rc;
  // reverse predictor:  g_in = g1 + gs - dt/2 J_D(U^n)^T gs
  return rev_stage<T>(c, DH_K_REV1, U, c->gs, g1, c->gs, gin, dt, 0.5);
}

extern "C" {

int dh_cfl_dt_async(dh_ctx* c, const void* U) {
  if (!c || !U) return fail(DH_ERR_ARG, "dh_cfl_dt: NULL argument%s");
  if (int drc = check_device(c, "dh_cfl_dt_async")) return drc;
  return c->dtype == DH_F32 ? cfl_launch<float>(c, U) : cfl_launch<double>(c, U);
}

int dh_poll_status(dh_ctx* c, double* dt_out) {
  if (!c) return fail(DH_ERR_ARG, "dh_poll_status: NULL context%s");
  DH_CUDA(cudaMemcpyAsync(c->result_host, c->result_dev, sizeof(CflResult), cudaMemcpyDeviceToHost, c->stream), "dh_poll_status: copy");
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_poll_status: synchronize");
  if (c->result_host->nonfinite) return fail(DH_ERR_NONFINITE, "dh_cfl_dt: non-finite input or wave speed%s");
  if (dt_out) *dt_out = c->result_host->dt;
  return DH_OK;
}

int dh_cfl_dt(dh_ctx* c, const void* U, double* dt_out) {
  if (!dt_out) return fail(DH_ERR_ARG, "dh_cfl_dt: NULL dt_out%s");
  int rc = dh_cfl_dt_async(c, U);
  if (rc) return rc;
  return dh_poll_status(c, dt_out);
}

int dh_step(dh_ctx* c, void* U, double dt) {
  if (!c || !U) return fail(DH_ERR_ARG, "dh_step: NULL argument%s");
  if (int drc = check_device(c, "dh_step")) return drc;
  if (!(dt > 0.0) || !isfinite(dt)) return fail(DH_ERR_ARG, "dh_step: dt must be finite and > 0%s");
  if (U == c->Us) return fail(DH_ERR_ARG, "dh_step: U aliases library scratch%s");
  return c->dtype == DH_F32 ? step_impl<float>(c, U, dt, false) : step_impl<double>(c, U, dt, false);
}

int dh_step_devdt(dh_ctx* c, void* U) {
  if (!c || !U) return fail(DH_ERR_ARG, "dh_step_devdt: NULL argument%s");
  if (int drc = check_device(c, "dh_step_devdt")) return drc;
  return c->dtype == DH_F32 ? step_impl<float>(c, U, 0.0, true) : step_impl<double>(c, U, 0.0, true);
}

int dh_step_vjp(dh_ctx* c, const void* U, double dt, const void* gout, void* gin) {
  if (!c || !U || !gout || !gin) return fail(DH_ERR_ARG, "dh_step_vjp: NULL argument%s");
  if (int drc = check_device(c, "dh_step_vjp")) return drc;
  if (!(dt > 0.0) || !isfinite(dt)) return fail(DH_ERR_ARG, "dh_step_vjp: dt must be finite and > 0%s");
  if (gin == U || gin == gout) return fail(DH_ERR_ARG, "dh_step_vjp: gU_in must not alias U or gU_out%s");
  return c->dtype == DH_F32 ? vjp_impl<float>(c, U, dt, gout, gin) : vjp_impl<double>(c, U, dt, gout, gin);
}

int dh_advance(dh_ctx* c, void* U, int nsteps, double* dt_last_out) {
  if (!c || !U || nsteps < 0) return fail(DH_ERR_ARG, "dh_advance: bad argument%s");
  if (int drc = check_device(c, "dh_advance")) return drc;
  if (U == c->Us) return fail(DH_ERR_ARG, "dh_advance: U aliases library scratch%s");
  const bool f32 = c->dtype == DH_F32;
  // From the second step on, the CFL pass runs on the candidates the previous last stage pushed (DH_OPT_FUSE_CFL)
  // (not with the cooling-time limit of Eq. 21: t_cool needs every cell, so the full pass runs anyway)
  const bool fuse = c->fuse_cfl && nsteps > 1 && c->kernel == 0 && !(c->cooling != 0 && c->c_cool > 0.0);
  if (fuse) {
    int rc = cand_alloc(c);
    if (rc) return rc;
  }
  c->cand_ok = 0;
  for (int s = 0; s < nsteps; ++s) {
    const bool use = fuse && s > 0 && c->cand_ok;
    int rc = f32 ? cfl_launch<float>(c, U, use) : cfl_launch<double>(c, U, use);
    if (rc) return rc;
    const bool push = fuse && s + 1 < nsteps;
    rc = f32 ? step_impl<float>(c, U, 0.0, true, push) : step_impl<double>(c, U, 0.0, true, push);
    if (rc) return rc;
  }
  c->cand_ok = 0;
  if (dt_last_out) return dh_poll_status(c, dt_last_out);
  return DH_OK;
}

int dh_cool_tmin(dh_ctx* c, const void* U, double* tcool_min_out, double* dt_hydro_out) {
  if (!c || !U || !tcool_min_out) return fail(DH_ERR_ARG, "dh_cool_tmin: NULL argument%s");
  if (int drc = check_device(c, "dh_cool_tmin")) return drc;
  int rc = c->dtype == DH_F32 ? cfl_launch<float>(c, U, false, true) : cfl_launch<double>(c, U, false, true);
  if (rc) return rc;
  rc = dh_poll_status(c, nullptr);
  if (rc) return rc;
  *tcool_min_out = c->result_host->tcool_min;
  if (dt_hydro_out) *dt_hydro_out = c->result_host->dt_hydro;
  return DH_OK;
}

int dh_set_cooling_table(dh_ctx* c, const double* log10_lambda, int n, double log10_t0, double dlog10_t) {
  if (!c || !log10_lambda) return fail(DH_ERR_ARG, "dh_set_cooling_table: NULL argument%s");
  if (int drc = check_device(c, "dh_set_cooling_table")) return drc;
  if (n < 2 || n > 256) return fail(DH_ERR_ARG, "dh_set_cooling_table: the table needs 2 .. 256 nodes%s");
  if (!(dlog10_t > 0.0) || !isfinite(dlog10_t) || !isfinite(log10_t0)) return fail(DH_ERR_ARG, "dh_set_cooling_table: node spacing must be finite and > 0%s");
  double h64[256];
  float h32[256];
  const double l2_10 = 3.321928094887362;           // held as log2 Lambda: one lg2 / ex2 pair evaluates the interpolant
  for (int k = 0; k < n; ++k) {
    if (!isfinite(log10_lambda[k])) return fail(DH_ERR_ARG, "dh_set_cooling_table: non-finite table value%s");
    h64[k] = log10_lambda[k] * l2_10;
    h32[k] = (float)h64[k];
  }
  int rc = lazy_alloc(c, &c->tab_dev, 256 * sizeof(double), "the cooling table");
  if (rc) return rc;
  rc = lazy_alloc(c, (void**)&c->tab_dev_d, 256 * sizeof(double), "the cooling table (double)");
  if (rc) return rc;
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_set_cooling_table: synchronize");      // kernels in flight may read the old table
  DH_CUDA(cudaMemcpy(c->tab_dev_d, h64, n * sizeof(double), cudaMemcpyHostToDevice), "dh_set_cooling_table: upload");
  if (c->dtype == DH_F32) DH_CUDA(cudaMemcpy(c->tab_dev, h32, n * sizeof(float), cudaMemcpyHostToDevice), "dh_set_cooling_table: upload");
  else DH_CUDA(cudaMemcpy(c->tab_dev, h64, n * sizeof(double), cudaMemcpyHostToDevice), "dh_set_cooling_table: upload");
  c->ntab = n; c->tab_log10t0 = log10_t0; c->tab_dlog10t = dlog10_t;
  return DH_OK;
}

}  // extern "C"

template <class T>
static int table_vjp_impl(dh_ctx* c, const void* U, double dt, const void* gout, double* gtab_host) {
  int rc = lazy_alloc(c, &c->U1, state_bytes(c), "the pre-cooling state");
  if (rc) return rc;
  rc = lazy_alloc(c, (void**)&c->tab_part, ((size_t)cool_table_blocks() + 1) * 256 * sizeof(double), "the table-gradient partial sums");
  if (rc) return rc;
  // the pre-cooling state of the step (nothing was stored by dh_step)
  if (c->integrator == 0) {
    rc = stage_launch<T>(c, DH_K_STAGE1, U, U, c->Us, dt, false, 0.5, false);
    if (rc) return rc;
    rc = stage_launch<T>(c, DH_K_STAGE2, c->Us, U, c->U1, dt, false, 1.0, false);
  } else {
    const void* last_in = nullptr;
    double w = 0.0;
    rc = rk_prefix<T>(c, U, dt, false, &last_in, &w);
    if (rc) return rc;
    rc = rk_last<T>(c, last_in, w, U, c->U1, dt, false, false, false);
  }
  if (rc) return rc;
  double* const res = c->tab_part + (size_t)cool_table_blocks() * 256;
  DH_CUDA(launch_cool_table_vjp<T>((const T*)c->U1, (const T*)gout, c->N, (T)dt, make_consts<T>(c), c->tab_part, res, c->stream),
          "dh_cool_table_vjp: kernel launch");
  c->launches += 2;
  DH_CUDA(cudaMemcpyAsync(gtab_host, res, c->ntab * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "dh_cool_table_vjp: copy");
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_cool_table_vjp: synchronize");
  return DH_OK;
}

extern "C" {

int dh_cool_table_vjp(dh_ctx* c, const void* U, double dt, const void* gU_out, double* gtab_out) {
  if (!c || !U || !gU_out || !gtab_out) return fail(DH_ERR_ARG, "dh_cool_table_vjp: NULL argument%s");
  if (int drc = check_device(c, "dh_cool_table_vjp")) return drc;
  if (!(dt > 0.0) || !isfinite(dt)) return fail(DH_ERR_ARG, "dh_cool_table_vjp: dt must be finite and > 0%s");
  if (!c->cooling || c->cool_law != 1 || c->ntab < 2) return fail(DH_ERR_ARG, "dh_cool_table_vjp: needs DH_OPT_COOLING = 1 and DH_OPT_COOL_LAW = 1%s");
  return c->dtype == DH_F32 ? table_vjp_impl<float>(c, U, dt, gU_out, gtab_out) : table_vjp_impl<double>(c, U, dt, gU_out, gtab_out);
}

int dh_cfl_stats(dh_ctx* c, unsigned long long* out) {
  if (!c || !out) return fail(DH_ERR_ARG, "dh_cfl_stats: NULL argument%s");
  out[0] = out[1] = out[2] = 0ull;
  if (!c->cand_stats) return DH_OK;
  DH_CUDA(cudaMemcpyAsync(out, c->cand_stats, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream), "dh_cfl_stats: copy");
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_cfl_stats: synchronize");
  return DH_OK;
}

int dh_adjoint(dh_ctx* c, void* U, void* gU, int nsteps, int every, double* dts_out) {
  if (!c || !U || !gU || nsteps < 0 || every < 1) return fail(DH_ERR_ARG, "dh_adjoint: bad argument%s");
  if (int drc = check_device(c, "dh_adjoint")) return drc;
  if (U == gU || U == c->Us || gU == c->Us) return fail(DH_ERR_ARG, "dh_adjoint: U and gU must be distinct caller arrays%s");
  if (nsteps == 0) return DH_OK;
  if (every > nsteps) every = nsteps;
  const size_t sb = state_bytes(c);
  const int nck = (nsteps + every - 1) / every;                 // checkpoints: states before steps 0, every, 2 every, ...
  const size_t need = (size_t)nck + (size_t)every + 1;          // + one segment of states + one cotangent
  if (c->adj_states && c->adj_count < need) {
    DH_CUDA(cudaStreamSynchronize(c->stream), "dh_adjoint: synchronize");
    cudaFree(c->adj_states);
    c->adj_states = nullptr;
  }
  if (!c->adj_states) {
    int rc = lazy_alloc(c, &c->adj_states, need * sb, "the checkpoints of dh_adjoint");
    if (rc) return rc;
    c->adj_count = need;
  }
  if (c->adj_dts_cap < nsteps) {
    DH_CUDA(cudaStreamSynchronize(c->stream), "dh_adjoint: synchronize");
    if (c->adj_dts_dev) cudaFree(c->adj_dts_dev);
    if (c->adj_dts_host) cudaFreeHost(c->adj_dts_host);
    c->adj_dts_dev = nullptr; c->adj_dts_host = nullptr; c->adj_dts_cap = 0;
    if (cudaMalloc((void**)&c->adj_dts_dev, 2 * (size_t)nsteps * 8) != cudaSuccess ||
        cudaMallocHost((void**)&c->adj_dts_host, 2 * (size_t)nsteps * 8) != cudaSuccess) {
      cudaGetLastError();
      return fail(DH_ERR_ALLOC, "dh_adjoint: allocation of the dt sequence failed%s");
    }
    c->adj_dts_cap = nsteps;
  }
  char* const base = (char*)c->adj_states;
  auto ckpt = [&](int i) { return (void*)(base + (size_t)i * sb); };
  auto seg = [&](int j) { return (void*)(base + ((size_t)nck + j) * sb); };
  void* gtmp = (void*)(base + ((size_t)nck + every) * sb);
  const bool f32 = c->dtype == DH_F32;
  // ---- forward sweep: checkpoints and the dt sequence (dt never visits the host inside the loop)
  for (int k = 0; k < nsteps; ++k) {
    if (k % every == 0) DH_CUDA(cudaMemcpyAsync(ckpt(k / every), U, sb, cudaMemcpyDeviceToDevice, c->stream), "dh_adjoint: checkpoint");
    int rc = f32 ? cfl_launch<float>(c, U) : cfl_launch<double>(c, U);
    if (rc) return rc;
    DH_CUDA(cudaMemcpyAsync(c->adj_dts_dev + k, &c->result_dev->dt, 8, cudaMemcpyDeviceToDevice, c->stream), "dh_adjoint: dt");
    DH_CUDA(cudaMemcpyAsync(c->adj_dts_dev + nsteps + k, &c->result_dev->nonfinite, 8, cudaMemcpyDeviceToDevice, c->stream), "dh_adjoint: flag");
    rc = f32 ? step_impl<float>(c, U, 0.0, true) : step_impl<double>(c, U, 0.0, true);
    if (rc) return rc;
  }
  DH_CUDA(cudaMemcpyAsync(c->adj_dts_host, c->adj_dts_dev, 2 * (size_t)nsteps * 8, cudaMemcpyDeviceToHost, c->stream), "dh_adjoint: dt sequence");
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_adjoint: synchronize");
  for (int k = 0; k < nsteps; ++k) {
    unsigned long long flag;
    memcpy(&flag, c->adj_dts_host + nsteps + k, 8);
    if (flag) return fail(DH_ERR_NONFINITE, "dh_adjoint: non-finite state in the forward sweep%s");
    if (dts_out) dts_out[k] = c->adj_dts_host[k];
  }
  // ---- reverse sweep, segment by segment: recompute the states before each step of the segment, then pull the
  //      cotangent back through the steps in reverse order
  void* g = gU;
  void* gn = gtmp;
  for (int ic = nck - 1; ic >= 0; --ic) {
    const int k0 = ic * every, len = (nsteps - k0 < every) ? nsteps - k0 : every;
    DH_CUDA(cudaMemcpyAsync(seg(0), ckpt(ic), sb, cudaMemcpyDeviceToDevice, c->stream), "dh_adjoint: segment start");
    for (int j = 1; j < len; ++j) {
      DH_CUDA(cudaMemcpyAsync(seg(j), seg(j - 1), sb, cudaMemcpyDeviceToDevice, c->stream), "dh_adjoint: segment copy");
      int rc = dh_step(c, seg(j), c->adj_dts_host[k0 + j - 1]);
      if (rc) return rc;
    }
    for (int j = len - 1; j >= 0; --j) {
      int rc = dh_step_vjp(c, seg(j), c->adj_dts_host[k0 + j], g, gn);
      if (rc) return rc;
      void* t = g; g = gn; gn = t;
    }
  }
  if (g != gU) DH_CUDA(cudaMemcpyAsync(gU, g, sb, cudaMemcpyDeviceToDevice, c->stream), "dh_adjoint: result copy");
  return DH_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ self-gravity
template <class T>
static int grav_source_impl(dh_ctx* c, void* U, const void* phi, double dt) {
  const double dx[3] = {c->L[0] / c->nx, c->L[1] / c->ny, c->L[2] / c->nz};
  DH_CUDA(launch_grav_source<T>((T*)U, (const T*)phi, c->nx, c->ny, c->nz, dx, (T)dt, nullptr, c->stream), "dh_gravity_source: kernel launch");
  c->launches += 1;
  return DH_OK;
}

template <class T>
static int grav_source_vjp_impl(dh_ctx* c, const void* U, const void* phi, double dt, const void* gout, void* gin, void* gphi) {
  int rc = lazy_alloc(c, &c->grav_gb, 3 * c->N * elem_size(c), "the acceleration cotangents");
  if (rc) return rc;
  const double dx[3] = {c->L[0] / c->nx, c->L[1] / c->ny, c->L[2] / c->nz};
  DH_CUDA(launch_grav_source_vjp<T>((const T*)U, (const T*)phi, (const T*)gout, (T*)gin, (T*)c->grav_gb, (T*)gphi, c->nx, c->ny, c->nz, dx, (T)dt, c->stream),
          "dh_gravity_source_vjp: kernel launch");
  c->launches += 2;
  return DH_OK;
}

static int grav_check(dh_ctx* c, dh_mg* mg, const char* who) {
  if (!c || !mg) return fail(DH_ERR_ARG, "%s: NULL context", who);
  if (int drc = check_device(c, who)) return drc;
  return DH_OK;
}

// phi of the incoming density into c->grav_phi (Eq. 27; the solver removes the mean of the right-hand side, reading A23)
template <class T>
static int grav_potential(dh_ctx* c, dh_mg* mg, const void* U, double four_pi_g, int ncycles) {
  int rc = lazy_alloc(c, &c->grav_phi, c->N * elem_size(c), "the gravitational potential");
  if (rc) return rc;
  rc = lazy_alloc(c, &c->grav_F, c->N * elem_size(c), "the Poisson right-hand side");
  if (rc) return rc;
  DH_CUDA(launch_grav_rhs<T>((const T*)U, (T*)c->grav_F, c->N, (T)four_pi_g, c->stream), "dh_step_gravity: right-hand side kernel");
  c->launches += 1;
  if (dh_mg_set_stream(mg, (void*)c->stream) != DH_OK) return fail(DH_ERR_ARG, "dh_step_gravity: %s", dh_last_error());
  if (dh_mg_solve(mg, c->grav_F, c->grav_phi, ncycles, nullptr) != DH_OK) return fail(DH_ERR_CUDA, "dh_step_gravity: Poisson solve: %s", dh_last_error());
  return DH_OK;
}

template <class T>
static int step_gravity_impl(dh_ctx* c, dh_mg* mg, void* U, double dt, double four_pi_g, int ncycles) {
  int rc = grav_potential<T>(c, mg, U, four_pi_g, ncycles);
  if (rc) return rc;
  rc = dh_step(c, U, dt);
  if (rc) return rc;
  return grav_source_impl<T>(c, U, c->grav_phi, dt);
}

template <class T>
static int step_gravity_vjp_impl(dh_ctx* c, dh_mg* mg, const void* U, double dt, double four_pi_g, int ncycles, const void* gout, void* gin) {
  int rc = lazy_alloc(c, &c->grav_U1, state_bytes(c), "the post-hydro state");
  if (rc) return rc;
  rc = lazy_alloc(c, &c->grav_g1, state_bytes(c), "the post-hydro cotangent");
  if (rc) return rc;
  rc = grav_potential<T>(c, mg, U, four_pi_g, ncycles);                       // recompute: nothing was stored
  if (rc) return rc;
  DH_CUDA(cudaMemcpyAsync(c->grav_U1, U, state_bytes(c), cudaMemcpyDeviceToDevice, c->stream), "dh_step_gravity_vjp: copy");
  rc = dh_step(c, c->grav_U1, dt);
  if (rc) return rc;
  // through the kick at the post-hydro state: cotangents of that state and of phi (into grav_F)
  rc = grav_source_vjp_impl<T>(c, c->grav_U1, c->grav_phi, dt, gout, c->grav_g1, c->grav_F);
  if (rc) return rc;
  // through the Poisson solve: another solve (Eqs. 46-48), result into grav_phi (the potential is dead)
  if (dh_mg_solve_vjp(mg, c->grav_F, c->grav_phi, ncycles, nullptr) != DH_OK) return fail(DH_ERR_CUDA, "dh_step_gravity_vjp: adjoint Poisson solve: %s", dh_last_error());
  // through the hydro step, then the density cotangent of the right-hand side F = 4 pi G rho
  rc = dh_step_vjp(c, U, dt, c->grav_g1, gin);
  if (rc) return rc;
  DH_CUDA(launch_grav_rhs_vjp<T>((const T*)c->grav_phi, (T*)gin, c->N, (T)four_pi_g, c->stream), "dh_step_gravity_vjp: right-hand side transpose");
  c->launches += 1;
  return DH_OK;
}

extern "C" {

int dh_gravity_source(dh_ctx* c, void* U, const void* phi, double dt) {
  if (!c || !U || !phi) return fail(DH_ERR_ARG, "dh_gravity_source: NULL argument%s");
  if (int drc = check_device(c, "dh_gravity_source")) return drc;
  if (!isfinite(dt)) return fail(DH_ERR_ARG, "dh_gravity_source: dt must be finite%s");
  return c->dtype == DH_F32 ? grav_source_impl<float>(c, U, phi, dt) : grav_source_impl<double>(c, U, phi, dt);
}

int dh_gravity_source_vjp(dh_ctx* c, const void* U, const void* phi, double dt, const void* gU_out, void* gU_in, void* gphi) {
  if (!c || !U || !phi || !gU_out || !gU_in || !gphi) return fail(DH_ERR_ARG, "dh_gravity_source_vjp: NULL argument%s");
  if (int drc = check_device(c, "dh_gravity_source_vjp")) return drc;
  if (!isfinite(dt)) return fail(DH_ERR_ARG, "dh_gravity_source_vjp: dt must be finite%s");
  if (gU_in == gU_out || gU_in == U) return fail(DH_ERR_ARG, "dh_gravity_source_vjp: gU_in must not alias gU_out or U%s");
  return c->dtype == DH_F32 ? grav_source_vjp_impl<float>(c, U, phi, dt, gU_out, gU_in, gphi) : grav_source_vjp_impl<double>(c, U, phi, dt, gU_out, gU_in, gphi);
}

int dh_step_gravity(dh_ctx* c, dh_mg* mg, void* U, double dt, double four_pi_g, int ncycles) {
  if (int rc = grav_check(c, mg, "dh_step_gravity")) return rc;
  if (!U || ncycles < 1) return fail(DH_ERR_ARG, "dh_step_gravity: bad argument%s");
  if (!(dt > 0.0) || !isfinite(dt) || !isfinite(four_pi_g)) return fail(DH_ERR_ARG, "dh_step_gravity: dt must be finite and > 0, four_pi_g finite%s");
  return c->dtype == DH_F32 ? step_gravity_impl<float>(c, mg, U, dt, four_pi_g, ncycles) : step_gravity_impl<double>(c, mg, U, dt, four_pi_g, ncycles);
}

int dh_step_gravity_vjp(dh_ctx* c, dh_mg* mg, const void* U, double dt, double four_pi_g, int ncycles, const void* gU_out, void* gU_in) {
  if (int rc = grav_check(c, mg, "dh_step_gravity_vjp")) return rc;
  if (!U || !gU_out || !gU_in || ncycles < 1) return fail(DH_ERR_ARG, "dh_step_gravity_vjp: bad argument%s");
  if (!(dt > 0.0) || !isfinite(dt) || !isfinite(four_pi_g)) return fail(DH_ERR_ARG, "dh_step_gravity_vjp: dt must be finite and > 0, four_pi_g finite%s");
  if (gU_in == U || gU_in == gU_out) return fail(DH_ERR_ARG, "dh_step_gravity_vjp: gU_in must not alias U or gU_out%s");
  return c->dtype == DH_F32 ? step_gravity_vjp_impl<float>(c, mg, U, dt, four_pi_g, ncycles, gU_out, gU_in)
                            : step_gravity_vjp_impl<double>(c, mg, U, dt, four_pi_g, ncycles, gU_out, gU_in);
}

}  // extern "C"

// dh_stream_host: a state that lives in HOST memory, every step reading it from there and writing it back (dh.h).
// Three streams: the link's two directions and the context's compute stream.  The state moves in z slabs; step n computes in
// device state n % 2:
//   H2D(n, k)   after D2H(n-1, k) has put slab k of the step's input into U_host          (h2d stream)
//   dt_n        from the resident copy of the same values (output of step n-1; the candidate CFL pass of dh_advance)
//   predictor   over the planes whose +-2 neighbours have arrived, as the slabs land (n >= 1; step 0 needs all of U for dt)
//   corrector   slab by slab in place, each followed by D2H(n, k)                          (d2h stream)
// so in the steady state both directions of the link are busy and the kernels hide behind them.  Results are those of
// dh_advance on a resident state bit for bit: the kernels do the same arithmetic per cell whatever z range a launch covers.
template <class T>
static int stream_host_impl(dh_ctx* c, void* U_host, int nsteps) {
  const size_t esz = sizeof(T), NP = (size_t)c->nx * c->ny, N = c->N;
  int S = c->stream_slab_opt > 0 ? c->stream_slab_opt : (c->nz + 31) / 32;
  if (S < 8) S = 8;
  if (S > c->nz) S = c->nz;
  const int ns = (c->nz + S - 1) / S;
  int rc = lazy_alloc(c, &c->Uhost_dev, state_bytes(c), "the device state of the host entry point");
  if (rc) return rc;
  rc = lazy_alloc(c, &c->Uhost_dev2, state_bytes(c), "the second device state of dh_stream_host");
  if (rc) return rc;
  if (!c->h2d_stream) DH_CUDA(cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking), "dh_stream_host: stream");
  if (!c->d2h_stream) DH_CUDA(cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking), "dh_stream_host: stream");
  if (c->ev_n < ns + 1) {
    for (int i = 0; i < 3 * c->ev_n; ++i) cudaEventDestroy(c->ev_slab[i]);
    free(c->ev_slab);
    c->ev_n = 0;
    c->ev_slab = (cudaEvent_t*)calloc((size_t)3 * (ns + 1), sizeof(cudaEvent_t));
    if (!c->ev_slab) return fail(DH_ERR_ALLOC, "dh_stream_host: out of host memory%s");
    for (int i = 0; i < 3 * (ns + 1); ++i) DH_CUDA(cudaEventCreateWithFlags(&c->ev_slab[i], cudaEventDisableTiming), "dh_stream_host: event");
    c->ev_n = ns + 1;
  }
  cudaEvent_t* const ev_in = c->ev_slab;
  cudaEvent_t* const ev_cmp = c->ev_slab + c->ev_n;
  cudaEvent_t* const ev_out = c->ev_slab + 2 * c->ev_n;
  cudaEvent_t const ev_sync = ev_in[ns];                       // entry / exit ordering against the context's stream
  void* const dev[2] = {c->Uhost_dev, c->Uhost_dev2};
  auto copy_slab = [&](void* dst, const void* src, int k, cudaMemcpyKind kind, cudaStream_t st) -> cudaError_t {
    const int z0 = k * S, cnt = (c->nz - z0 < S) ? c->nz - z0 : S;
    for (int f = 0; f < 5; ++f) {
      const size_t off = ((size_t)f * N + (size_t)z0 * NP) * esz;
      cudaError_t e = cudaMemcpyAsync((char*)dst + off, (const char*)src + off, (size_t)cnt * NP * esz, kind, st);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  };
  // work queued earlier on the context's stream may still use the device states
  DH_CUDA(cudaEventRecord(ev_sync, c->stream), "dh_stream_host: event record");
  DH_CUDA(cudaStreamWaitEvent(c->h2d_stream, ev_sync, 0), "dh_stream_host: stream wait");
  DH_CUDA(cudaStreamWaitEvent(c->d2h_stream, ev_sync, 0), "dh_stream_host: stream wait");

  const bool split_cool = c->cooling != 0 && (c->cool_mode != 0 || c->cool_nsub > 1 || c->cool_law != 0);
  const bool fused_cool = c->cooling != 0 && !split_cool;
  const bool ranges = fused_ok(c) && c->integrator == 0 && !split_cool;        // else: whole-grid launches, only the copies overlap
  const bool fuse = c->fuse_cfl && nsteps > 1 && c->kernel == 0 && !(c->cooling != 0 && c->c_cool > 0.0);
  if (fuse) {
    rc = cand_alloc(c);
    if (rc) return rc;
  }
  c->cand_ok = 0;
  for (int n = 0; n < nsteps; ++n) {
    void* const Ud = dev[n & 1];
    for (int k = 0; k < ns; ++k) {
      if (n > 0) DH_CUDA(cudaStreamWaitEvent(c->h2d_stream, ev_out[k], 0), "dh_stream_host: stream wait");
      DH_CUDA(copy_slab(Ud, U_host, k, cudaMemcpyHostToDevice, c->h2d_stream), "dh_stream_host: H2D");
      DH_CUDA(cudaEventRecord(ev_in[k], c->h2d_stream), "dh_stream_host: event record");
    }
    const bool push = fuse && n + 1 < nsteps;
    if (n == 0) {
      DH_CUDA(cudaStreamWaitEvent(c->stream, ev_in[ns - 1], 0), "dh_stream_host: stream wait");
      rc = cfl_launch<T>(c, Ud, false);
    } else {
      rc = cfl_launch<T>(c, dev[(n & 1) ^ 1], fuse && c->cand_ok);
    }
    if (rc) return rc;
    if (ranges) {
      StageExtra x;
      if (n == 0) {
        rc = stage_launch<T>(c, DH_K_STAGE1, Ud, Ud, c->Us, 0.0, true, 0.5, false);
        if (rc) return rc;
      } else {
        int done = 2;                                           // planes [2, done) of U* are launched
        for (int k = 0; k < ns; ++k) {
          DH_CUDA(cudaStreamWaitEvent(c->stream, ev_in[k], 0), "dh_stream_host: stream wait");
          const int landed = (k + 1) * S < c->nz ? (k + 1) * S : c->nz;
          const int hi = (k == ns - 1) ? c->nz + 2 : landed - 2;   // the last launch wraps around: planes nz-2, nz-1, 0, 1
          if (hi <= done) continue;
          x.zbeg = done; x.zcnt = hi - done;
          rc = stage_launch<T>(c, DH_K_STAGE1, Ud, Ud, c->Us, 0.0, true, 0.5, false, false, x);
          if (rc) return rc;
          done = hi;
        }
      }
      bool pushed = true;
      for (int k = 0; k < ns; ++k) {
        x.zbeg = k * S; x.zcnt = (c->nz - k * S < S) ? c->nz - k * S : S;
        rc = stage_launch<T>(c, DH_K_STAGE2, c->Us, Ud, Ud, 0.0, true, 1.0, fused_cool, push, x);
        if (rc) return rc;
        pushed = pushed && c->cand_ok;
        DH_CUDA(cudaEventRecord(ev_cmp[k], c->stream), "dh_stream_host: event record");
      }
      c->cand_ok = pushed ? 1 : 0;
    } else {
      DH_CUDA(cudaStreamWaitEvent(c->stream, ev_in[ns - 1], 0), "dh_stream_host: stream wait");
      rc = step_impl<T>(c, Ud, 0.0, true, push);
      if (rc) return rc;
      DH_CUDA(cudaEventRecord(ev_cmp[0], c->stream), "dh_stream_host: event record");
    }
    for (int k = 0; k < ns; ++k) {
      DH_CUDA(cudaStreamWaitEvent(c->d2h_stream, ev_cmp[ranges ? k : 0], 0), "dh_stream_host: stream wait");
      DH_CUDA(copy_slab(U_host, Ud, k, cudaMemcpyDeviceToHost, c->d2h_stream), "dh_stream_host: D2H");
      DH_CUDA(cudaEventRecord(ev_out[k], c->d2h_stream), "dh_stream_host: event record");
    }
  }
  c->cand_ok = 0;
  DH_CUDA(cudaEventRecord(ev_sync, c->d2h_stream), "dh_stream_host: event record");
  DH_CUDA(cudaStreamWaitEvent(c->stream, ev_sync, 0), "dh_stream_host: stream wait");
  return DH_OK;
}

extern "C" {

int dh_stream_host(dh_ctx* c, void* U_host, int nsteps, double* dt_last_out) {
  if (!c || !U_host || nsteps < 0) return fail(DH_ERR_ARG, "dh_stream_host: bad argument%s");
  if (int drc = check_device(c, "dh_stream_host")) return drc;
  if (nsteps > 0) {
    int rc = c->dtype == DH_F32 ? stream_host_impl<float>(c, U_host, nsteps) : stream_host_impl<double>(c, U_host, nsteps);
    if (rc) return rc;
  }
  return dh_poll_status(c, dt_last_out);
}

int dh_run_host(dh_ctx* c, void* U_host, int nsteps, double* dt_last_out) {
  if (!c || !U_host || nsteps < 0) return fail(DH_ERR_ARG, "dh_run_host: bad argument%s");
  if (int drc = check_device(c, "dh_run_host")) return drc;
  int rc = lazy_alloc(c, &c->Uhost_dev, state_bytes(c), "the device state of the host entry point");
  if (rc) return rc;
  DH_CUDA(cudaMemcpyAsync(c->Uhost_dev, U_host, state_bytes(c), cudaMemcpyHostToDevice, c->stream), "dh_run_host: H2D");
  rc = dh_advance(c, c->Uhost_dev, nsteps, nullptr);
  if (rc) return rc;
  DH_CUDA(cudaMemcpyAsync(U_host, c->Uhost_dev, state_bytes(c), cudaMemcpyDeviceToHost, c->stream), "dh_run_host: D2H");
  return dh_poll_status(c, dt_last_out);
}

int dh_step_vjp_host(dh_ctx* c, const void* U_host, double dt, const void* gout_host, void* gin_host) {
  if (!c || !U_host || !gout_host || !gin_host) return fail(DH_ERR_ARG, "dh_step_vjp_host: NULL argument%s");
  if (int drc = check_device(c, "dh_step_vjp_host")) return drc;
  int rc = lazy_alloc(c, &c->Uhost_dev, state_bytes(c), "the device state of the host entry point");
  if (rc) return rc;
  rc = lazy_alloc(c, &c->gA, state_bytes(c), "the device cotangent (in)");
  if (rc) return rc;
  rc = lazy_alloc(c, &c->gB, state_bytes(c), "the device cotangent (out)");
  if (rc) return rc;
  DH_CUDA(cudaMemcpyAsync(c->Uhost_dev, U_host, state_bytes(c), cudaMemcpyHostToDevice, c->stream), "dh_step_vjp_host: H2D");
  DH_CUDA(cudaMemcpyAsync(c->gA, gout_host, state_bytes(c), cudaMemcpyHostToDevice, c->stream), "dh_step_vjp_host: H2D");
  rc = dh_step_vjp(c, c->Uhost_dev, dt, c->gA, c->gB);
  if (rc) return rc;
  DH_CUDA(cudaMemcpyAsync(gin_host, c->gB, state_bytes(c), cudaMemcpyDeviceToHost, c->stream), "dh_step_vjp_host: D2H");
  DH_CUDA(cudaStreamSynchronize(c->stream), "dh_step_vjp_host: synchronize");
  return DH_OK;
}

}  // extern "C"
