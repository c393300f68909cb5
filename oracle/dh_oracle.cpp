// ORACLE — test infrastructure only (see dh_oracle.hpp).  C entry points for oracle/oracle.py.
// Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC dh_oracle.cpp -o liboracle.so
#include "dh_oracle.hpp"

#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

using namespace dho;

static Grid mkgrid(int nx, int ny, int nz) {
  Grid g;
  g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
  return g;
}

extern "C" {

int dho_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void dho_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// dtype: 0 = float32 array, 1 = float64 array.  The recipe runs in that type.
int dho_cfl_dt(int nx, int ny, int nz, const Params* p, double cfl, int dtype, const void* U,
               double* dt_out, double* smax_out) {
  Grid g = mkgrid(nx, ny, nz);
  if (dtype == 0) return cfl_dt<float>(g, *p, cfl, (const float*)U, dt_out, smax_out);
  return cfl_dt<double>(g, *p, cfl, (const double*)U, dt_out, smax_out);
}

int dho_prims(int nx, int ny, int nz, const Params* p, const double* U, double* W) {
  compute_prims<double>(mkgrid(nx, ny, nz), *p, U, W);
  return 0;
}

int dho_flux_divergence(int nx, int ny, int nz, const Params* p, const double* U, double* D) {
  flux_divergence<double>(mkgrid(nx, ny, nz), *p, U, D);
  return 0;
}

int dho_step(int nx, int ny, int nz, const Params* p, const double* U, double dt, double* Uout) {
  step<double>(mkgrid(nx, ny, nz), *p, U, dt, Uout);
  return 0;
}

// exact JVP of the full step by pushing one-slot dual numbers through the very same step<S>()
int dho_step_jvp(int nx, int ny, int nz, const Params* p, const double* U, const double* V, double dt,
                 double* Uout, double* dUout) {
  Grid g = mkgrid(nx, ny, nz);
  const size_t M = 5 * g.N();
  std::vector<Dual<1>> u(M), o(M);
  for (size_t c = 0; c < M; ++c) { u[c].v = U[c]; u[c].d[0] = V[c]; }
  step<Dual<1>>(g, *p, u.data(), dt, o.data());
  for (size_t c = 0; c < M; ++c) { Uout[c] = o[c].v; dUout[c] = o[c].d[0]; }
  return 0;
}

int dho_step_vjp(int nx, int ny, int nz, const Params* p, const double* U, double dt, const double* gout,
                 double* gin) {
  step_vjp(mkgrid(nx, ny, nz), *p, U, dt, gout, gin);
  return 0;
}

// gU = -tau J_D(U)^T gV   (one stage; for unit tests)
int dho_stage_vjp(int nx, int ny, int nz, const Params* p, const double* U, double tau, const double* gV,
                  double* gU) {
  Grid g = mkgrid(nx, ny, nz);
  std::memset(gU, 0, sizeof(double) * 5 * g.N());
  stage_vjp_accumulate(g, *p, U, tau, gV, gU);
  return 0;
}

int dho_cooling(long long N, const Params* p, double dt, const double* U, double* Uout) {
  for (long long c = 0; c < N; ++c) {
    double u[5], o[5];
    for (int f = 0; f < 5; ++f) u[f] = U[f * N + c];
    cool(u, dt, *p, p->tab, o);
    for (int f = 0; f < 5; ++f) Uout[f * N + c] = o[f];
  }
  return 0;
}

// batch of n independent Riemann problems; WL, WR, F are [5][n] (rho, vx, vy, vz, P)
int dho_riemann(long long n, const Params* p, int axis, const double* WL, const double* WR, double* F) {
  for (long long c = 0; c < n; ++c) {
    double l[5], r[5], f[5];
    for (int q = 0; q < 5; ++q) { l[q] = WL[q * n + c]; r[q] = WR[q * n + c]; }
    riemann(l, r, axis, *p, f);
    for (int q = 0; q < 5; ++q) F[q * n + c] = f[q];
  }
  return 0;
}

// reconstruction along one periodic line: W is [5][n]; WL/WR[.][i] are the states at face i+1/2
int dho_reconstruct(int n, const Params* p, const double* W, double* WL, double* WR) {
  for (int i = 0; i < n; ++i) {
    double a[5], b[5], c[5], d[5], l[5], r[5];
    for (int q = 0; q < 5; ++q) {
      a[q] = W[q * n + wrap(i - 1, n)]; b[q] = W[q * n + i];
      c[q] = W[q * n + wrap(i + 1, n)]; d[q] = W[q * n + wrap(i + 2, n)];
    }
    face_states(a, b, c, d, *p, l, r);
    for (int q = 0; q < 5; ++q) { WL[q * n + i] = l[q]; WR[q * n + i] = r[q]; }
  }
  return 0;
}

double dho_limiter(double a, double b, int kind) { return limiter<double>(a, b, kind); }

// Eqs. 20-21: min_x t_cool(x) in double, and the limited dt compared in the array's type
int dho_cool_dt(int nx, int ny, int nz, const Params* p, int dtype, const void* U, double dt_hydro, double c_cool,
                double dt_max, double* tmin_out, double* dt_out) {
  Grid g = mkgrid(nx, ny, nz);
  double tmin = dtype == 0 ? t_cool_min<float>(g, *p, (const float*)U) : t_cool_min<double>(g, *p, (const double*)U);
  *tmin_out = tmin;
  *dt_out = dtype == 0 ? limited_dt<float>(dt_hydro, tmin, c_cool, dt_max) : limited_dt<double>(dt_hydro, tmin, c_cool, dt_max);
  return 0;
}

// decision margins of one flux-divergence evaluation at U: M is [4][nz][ny][nx] (see dh_oracle.hpp)
int dho_decision_margins(int nx, int ny, int nz, const Params* p, const double* U, double* M) {
  decision_margins(mkgrid(nx, ny, nz), *p, U, M);
  return 0;
}

// conditioning of the limiter's derivative at U: C is [3][nz][ny][nx] (van Leer; zero for minmod / MC)
int dho_limiter_conditioning(int nx, int ny, int nz, const Params* p, const double* U, double* C) {
  limiter_conditioning(mkgrid(nx, ny, nz), *p, U, C);
  return 0;
}

// margins of the compares of cool() at the pre-cooling state U1: M is [nz][ny][nx]
int dho_cooling_margins(int nx, int ny, int nz, const Params* p, double dt, const double* U1, double* M) {
  cooling_margins(mkgrid(nx, ny, nz), *p, dt, U1, M);
  return 0;
}

// Lambda-side pieces for the pins: Edot(E_th, rho) of cool_rate() and the tabulated Lambda_CIE(T) of Eq. 19
double dho_cool_rate(const Params* p, double Eth, double rho) { return cool_rate<double>(Eth, rho, *p, p->tab); }
double dho_lambda_table(const Params* p, double T) { return lambda_table<double>(T, *p, p->tab); }

// gradient of sum(gout_E * E_out) with respect to the table nodes, at the pre-cooling state U1 (ntab <= 32)
int dho_cooling_table_vjp(int nx, int ny, int nz, const Params* p, double dt, const double* U1, const double* gout, double* gtab) {
  return cooling_table_vjp(mkgrid(nx, ny, nz), *p, dt, U1, gout, gtab);
}

// the pre-cooling state of a step (what cooling_vjp / cooling_table_vjp are evaluated at): the step with cooling off
int dho_step_nocool(int nx, int ny, int nz, const Params* p, const double* U, double dt, double* Uout) {
  Params q = *p;
  q.cooling = 0;
  step<double>(mkgrid(nx, ny, nz), q, U, dt, Uout);
  return 0;
}

}  // extern "C"

