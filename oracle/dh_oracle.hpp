// ORACLE — test infrastructure only.
//
// Plain, slow, obviously-correct CPU implementation of the hot path of arxiv/paper_2512_13403
// ("diffhydro"): one explicit step of the 3D compressible Euler finite-volume update on a uniform
// periodic Cartesian grid, its CFL time step, the optional pointwise cooling source, and the
// discrete adjoint (VJP) of the step.  Written from PAPER.md; it shares no code with the CUDA path
// under paper_2512_13403_b200/ and neither imports the other.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call anything in oracle/.
//
// Everything is templated on the scalar type S so that the *same* literal transcription of the
// scheme runs on double (forward), on dual numbers (exact JVP, and local Jacobians for the VJP)
// and on float (the dt recipe, which must be reproduced bit-for-bit by the GPU).
//
// Citations are PAPER.md:<line> (section / equation).  Readings of silent or ambiguous points are
// the A1..A16 rows of SURVEY.md §8(c); they are restated in DESIGN.md.
//
// Layout: U[f][k][j][i], f in {0:rho, 1:rho*vx, 2:rho*vy, 3:rho*vz, 4:E}  (Eq. 2;
// PAPER.md:96-104), i (x) fastest, periodic in all three directions.
#pragma once
#include <cmath>
#include <limits>
#include <cstddef>
#include <vector>

namespace dho {

// ------------------------------------------------------------------------------------------------
// Parameters (plain C struct; mirrored field by field in oracle/oracle.py)
// ------------------------------------------------------------------------------------------------
struct Params {
  double gamma;       // adiabatic index
  double dx[3];       // cell sizes Delta x_a (Eq. A4)
  double rho_floor;   // floors used only inside prim() (reading A6)
  double p_floor;
  int limiter;        // 0 minmod (A4), 1 van Leer, 2 MC, 3 piecewise-constant
  int riemann;        // 0 HLLC, 1 HLL, 2 Rusanov/LF
  int integrator;     // 0 predictor/corrector A6-A7, 1 Heun, 2 SSPRK3
  int cooling;        // 0 off, 1 on; which update: cool_mode / cool_nsub below
  double lambda0;     // Lambda(T) = lambda0 * T^alpha (reading A10)
  double alpha;
  double t_floor;     // temperature floor, Eq. 24 with R=1
  int cool_mode;      // 0: Euler + floor of Eq. 23, sub-cycled; 1: trapezoid of Eq. 22, reading A20
  int cool_nsub;      // N_sub >= 1 substeps of size dt / N_sub in mode 0
  // --- the two-branch law of Eqs. 17-19 and the masked choice of integrator ---
  int cool_law;       // 0: Lambda = lambda0 T^alpha, Gamma = 0 (reading A10); 1: Eq. 17: Koyama-Inutsuka fit + uniform heating below
                      //    t_switch, tabulated Lambda_CIE above it (reading A25)
  double t_switch;    // the 10^4 K of Eq. 17, in code units
  double lambda1, alpha1, lambda2, alpha2;   // Eq. 18: Lambda_KI = lambda1 T^alpha1 + lambda2 T^alpha2
  double gamma0;      // uniform heating rate Gamma_0 for T < t_switch; enters as n_H Gamma (Eq. 20)
  const double* tab;  // log10 Lambda_CIE at the nodes log10 T = tab_logT0 + k tab_dlogT, k = 0 .. ntab-1 (Eq. 19)
  int ntab;
  double tab_logT0, tab_dlogT;
  double f_sub;       // cool_mode 2: a cell is sub-cycled (Eq. 23) when dt |Edot(T^n)| > f_sub |E_th^n|, else Eq. 22 (reading A26)
};

// ------------------------------------------------------------------------------------------------
// Dual numbers with N derivative slots (forward-mode AD; exact to rounding)
// ------------------------------------------------------------------------------------------------
template <int N>
struct Dual {
  double v;
  double d[N];
  Dual() : v(0.0) { for (int i = 0; i < N; ++i) d[i] = 0.0; }
  Dual(double x) : v(x) { for (int i = 0; i < N; ++i) d[i] = 0.0; }
};

template <int N> inline Dual<N> operator+(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v + b.v; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
template <int N> inline Dual<N> operator-(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v - b.v; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
template <int N> inline Dual<N> operator-(const Dual<N>& a) { Dual<N> r; r.v = -a.v; for (int i = 0; i < N; ++i) r.d[i] = -a.d[i]; return r; }
template <int N> inline Dual<N> operator*(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v * b.v; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
template <int N> inline Dual<N> operator/(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v / b.v; for (int i = 0; i < N; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v; return r; }
template <int N> inline Dual<N> operator+(const Dual<N>& a, double b) { Dual<N> r = a; r.v += b; return r; }
template <int N> inline Dual<N> operator+(double a, const Dual<N>& b) { return b + a; }
template <int N> inline Dual<N> operator-(const Dual<N>& a, double b) { Dual<N> r = a; r.v -= b; return r; }
template <int N> inline Dual<N> operator-(double a, const Dual<N>& b) { return (-b) + a; }
template <int N> inline Dual<N> operator*(const Dual<N>& a, double b) { Dual<N> r; r.v = a.v * b; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] * b; return r; }
template <int N> inline Dual<N> operator*(double a, const Dual<N>& b) { return b * a; }
template <int N> inline Dual<N> operator/(const Dual<N>& a, double b) { Dual<N> r; r.v = a.v / b; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] / b; return r; }
template <int N> inline Dual<N> operator/(double a, const Dual<N>& b) { return Dual<N>(a) / b; }

// value of a scalar (the quantity every branch looks at: the a.e. derivative follows the branch
// actually taken, reading A7)
inline double val(double a) { return a; }
inline double val(float a) { return (double)a; }
template <int N> inline double val(const Dual<N>& a) { return a.v; }

inline double ssqrt(double a) { return std::sqrt(a); }
inline float ssqrt(float a) { return std::sqrt(a); }
template <int N> inline Dual<N> ssqrt(const Dual<N>& a) { Dual<N> r; r.v = std::sqrt(a.v); for (int i = 0; i < N; ++i) r.d[i] = a.d[i] / (2.0 * r.v); return r; }

inline double slog10(double a) { return std::log10(a); }
template <int N> inline Dual<N> slog10(const Dual<N>& a) { Dual<N> r; r.v = std::log10(a.v); for (int i = 0; i < N; ++i) r.d[i] = a.d[i] / (a.v * 2.302585092994045684); return r; }
inline double spow10(double a) { return std::pow(10.0, a); }
template <int N> inline Dual<N> spow10(const Dual<N>& a) { Dual<N> r; r.v = std::pow(10.0, a.v); for (int i = 0; i < N; ++i) r.d[i] = 2.302585092994045684 * r.v * a.d[i]; return r; }

inline double spow(double a, double p) { return std::pow(a, p); }
template <int N> inline Dual<N> spow(const Dual<N>& a, double p) { Dual<N> r; r.v = std::pow(a.v, p); double g = (a.v > 0.0) ? p * std::pow(a.v, p - 1.0) : 0.0; for (int i = 0; i < N; ++i) r.d[i] = g * a.d[i]; return r; }

// min/max: ties -> first argument (reading A7)
template <class S> inline S smax(const S& a, const S& b) { return (val(a) >= val(b)) ? a : b; }
template <class S> inline S smin(const S& a, const S& b) { return (val(a) <= val(b)) ? a : b; }
template <class S> inline S sabs(const S& a) { return (val(a) >= 0.0) ? a : S(-a); }

// ------------------------------------------------------------------------------------------------
// Step 1 — primitive conversion  W = (rho, v, P),  P = (gamma-1)(E - rho|v|^2/2)   (
// PAPER.md:811).  Floors act only here, conserved arrays are never modified (reading A6).
// ------------------------------------------------------------------------------------------------
template <class S>
inline void prim(const S U[5], const Params& p, S W[5]) {
  S rho = smax(U[0], S(p.rho_floor));
  W[0] = rho;
  W[1] = U[1] / rho;
  W[2] = U[2] / rho;
  W[3] = U[3] / rho;
  S m2 = U[1] * U[1] + U[2] * U[2] + U[3] * U[3];
  S P = (p.gamma - 1.0) * (U[4] - 0.5 * m2 / rho);
  W[4] = smax(P, S(p.p_floor));
}

// ------------------------------------------------------------------------------------------------
// Step 2 — slope limiters for Eq. A1; the menu is PAPER.md:820, formulas are the
// textbook ones (reading A4).  a = W_{i+1}-W_i, b = W_i-W_{i-1}.
// ------------------------------------------------------------------------------------------------
template <class S>
inline S limiter(const S& a, const S& b, int kind) {
  if (kind == 3) return S(0.0);                      // piecewise constant
  if (val(a) * val(b) <= 0.0) return S(0.0);         // extremum: zero slope (all limiters)
  if (kind == 0) {                                   // minmod; |a|==|b| -> a (A7)
    return (std::fabs(val(a)) <= std::fabs(val(b))) ? a : b;
  } else if (kind == 1) {                            // van Leer: harmonic mean
    return 2.0 * a * b / (a + b);
  } else {                                           // MC: minmod(2a, 2b, (a+b)/2)
    S c = 0.5 * (a + b);
    S a2 = 2.0 * a, b2 = 2.0 * b;
    S m = (std::fabs(val(a2)) <= std::fabs(val(b2))) ? a2 : b2;
    return (std::fabs(val(m)) <= std::fabs(val(c))) ? m : c;
  }
}

// Euler flux along axis ax of a primitive state, and its conserved vector.
template <class S>
inline void phys_flux(const S W[5], int ax, double gamma, S Ucons[5], S F[5]) {
  S rho = W[0], P = W[4];
  S un = W[1 + ax];
  S E = P / (gamma - 1.0) + 0.5 * rho * (W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
  Ucons[0] = rho;
  Ucons[1] = rho * W[1];
  Ucons[2] = rho * W[2];
  Ucons[3] = rho * W[3];
  Ucons[4] = E;
  F[0] = rho * un;
  F[1] = rho * un * W[1];
  F[2] = rho * un * W[2];
  F[3] = rho * un * W[3];
  F[1 + ax] = F[1 + ax] + P;
  F[4] = un * (E + P);
}

// ------------------------------------------------------------------------------------------------
// Step 3 — Riemann flux at a face from left/right primitive states.
// Wave speeds: Eq. A3, c_s^2 = gamma P / rho.  The rest of HLLC is
// not printed in the paper (it defers to HL25); textbook HLLC with the pressure-based contact
// speed and the F_K + S_K (U*_K - U_K) form is used (reading A3).  Select order and >=/<= as in
// SURVEY.md §8(c) step 3 (reading A7).
// ------------------------------------------------------------------------------------------------
template <class S>
inline void riemann(const S L[5], const S R[5], int ax, const Params& p, S F[5]) {
  const double g = p.gamma;
  S uL = L[1 + ax], uR = R[1 + ax];
  S cL = ssqrt(g * L[4] / L[0]);
  S cR = ssqrt(g * R[4] / R[0]);
  S SL = smin(S(uL - cL), S(uR - cR));   // Eq. A3
  S SR = smax(S(uL + cL), S(uR + cR));
  S UL[5], UR[5], FL[5], FR[5];
  phys_flux(L, ax, g, UL, FL);
  phys_flux(R, ax, g, UR, FR);

  if (p.riemann == 2) {  // Rusanov / local Lax-Friedrichs
    S a = smax(sabs(SL), sabs(SR));
    for (int f = 0; f < 5; ++f) F[f] = 0.5 * (FL[f] + FR[f]) - 0.5 * a * (UR[f] - UL[f]);
    return;
  }
  if (val(SL) >= 0.0) { for (int f = 0; f < 5; ++f) F[f] = FL[f]; return; }
  if (val(SR) <= 0.0) { for (int f = 0; f < 5; ++f) F[f] = FR[f]; return; }
  if (p.riemann == 1) {  // two-wave HLL
    for (int f = 0; f < 5; ++f) F[f] = (SR * FL[f] - SL * FR[f] + SL * SR * (UR[f] - UL[f])) / (SR - SL);
    return;
  }
  // HLLC
  S rhoL = L[0], rhoR = R[0], PL = L[4], PR = R[4];
  S Sstar = (PR - PL + rhoL * uL * (SL - uL) - rhoR * uR * (SR - uR)) /
            (rhoL * (SL - uL) - rhoR * (SR - uR));
  const bool left = (val(Sstar) >= 0.0);
  const S* W = left ? L : R;
  const S* UK = left ? UL : UR;
  const S* FK = left ? FL : FR;
  S SK = left ? SL : SR;
  S rhoK = W[0], uK = W[1 + ax], PK = W[4];
  S fac = rhoK * (SK - uK) / (SK - Sstar);
  S Ustar[5];
  Ustar[0] = fac;
  Ustar[1] = fac * W[1];
  Ustar[2] = fac * W[2];
  Ustar[3] = fac * W[3];
  Ustar[1 + ax] = fac * Sstar;
  Ustar[4] = fac * (UK[4] / rhoK + (Sstar - uK) * (Sstar + PK / (rhoK * (SK - uK))));
  for (int f = 0; f < 5; ++f) F[f] = FK[f] + SK * (Ustar[f] - UK[f]);
}

// ------------------------------------------------------------------------------------------------
// Steps 2+3 for one face i+1/2 from the four cells i-1, i, i+1, i+2 along the axis:
// Delta W_i = lim(W_{i+1}-W_i, W_i-W_{i-1})                        (Eq. A1)
// W^L = W_i + Delta W_i / 2,  W^R = W_{i+1} - Delta W_{i+1} / 2    (Eq. A2)
// ------------------------------------------------------------------------------------------------
template <class S>
inline void face_states(const S Wm1[5], const S W0[5], const S Wp1[5], const S Wp2[5],
                        const Params& p, S WL[5], S WR[5]) {
  for (int c = 0; c < 5; ++c) {
    S d0 = limiter(S(Wp1[c] - W0[c]), S(W0[c] - Wm1[c]), p.limiter);
    S d1 = limiter(S(Wp2[c] - Wp1[c]), S(Wp1[c] - W0[c]), p.limiter);
    WL[c] = W0[c] + 0.5 * d0;
    WR[c] = Wp1[c] - 0.5 * d1;
  }
}

template <class S>
inline void face_flux(const S Wm1[5], const S W0[5], const S Wp1[5], const S Wp2[5], int ax,
                      const Params& p, S F[5]) {
  S WL[5], WR[5];
  face_states(Wm1, W0, Wp1, Wp2, p, WL, WR);
  riemann(WL, WR, ax, p, F);
}

// ------------------------------------------------------------------------------------------------
// Step 6 — pointwise cooling, applied once after the hydro update and changing only E.
// Code units n = rho, T = P/rho, Gamma = 0, Lambda = lambda0 T^alpha (reading A10), so
//   Edot(E_th) = -rho^2 lambda0 max(T, 0)^alpha,   T = (gamma-1) E_th / rho.
// cool_mode 0: the sub-cycled update of Eq. 23: N_sub substeps delta t = dt / N_sub,
//   E_th^{k+1} = max(E_floor, E_th^k + Edot(T^k) delta t), T^k re-evaluated every substep; N_sub = 1 is reading A9.
//   (The "maximum fractional change" limiter the paper mentions without a formula is not applied, reading A9.)
// cool_mode 1: the trapezoid of Eq. 22: E_th^{n+1} = E_th^n + dt/2 [Edot(T^n) + Edot(T^pred)]; the
//   paper does not define T^pred: reading A20 takes the temperature of the Euler-predicted, floored energy
//   E_pred = max(E_floor, E_th^n + Edot(T^n) dt), and floors the result by Eq. 24 as well.
// Floor: Eq. 24 with R = 1.
// ------------------------------------------------------------------------------------------------
// Lambda_CIE(T) of Eq. 19: linear interpolation in log10 T - log10 Lambda between the table nodes.
// Reading A25: outside the table the end values are held (T >= t_switch >= first node in every use).
template <class S>
inline S lambda_table(const S& T, const Params& p, const S* tab) {
  S u = (slog10(T) - p.tab_logT0) / p.tab_dlogT;
  int k = (int)std::floor(val(u));
  if (k < 0) k = 0;
  if (k > p.ntab - 2) k = p.ntab - 2;
  S w = u - (double)k;
  if (val(w) < 0.0) w = S(0.0);
  if (val(w) > 1.0) w = S(1.0);
  return spow10(S(tab[k] + w * (tab[k + 1] - tab[k])));
}

// Edot = n_H Gamma - n_H^2 Lambda (Eqs. 15, 20 with chi = 1) in code units n_H = rho, T = (gamma-1) E_th / rho
template <class S>
inline S cool_rate(const S& Eth, const S& rho, const Params& p, const S* tab) {
  S T = (p.gamma - 1.0) * Eth / rho;
  S Tpos = smax(T, S(0.0));
  if (p.cool_law == 0) return -1.0 * rho * rho * p.lambda0 * spow(Tpos, p.alpha);
  if (val(T) < p.t_switch)                                   // Eq. 17, lower branch: Eq. 18 and Gamma_0
    return rho * p.gamma0 - rho * rho * (p.lambda1 * spow(Tpos, p.alpha1) + p.lambda2 * spow(Tpos, p.alpha2));
  return -1.0 * rho * rho * lambda_table(T, p, tab);         // upper branch: Eq. 19, no heating
}

// the table as scalars of type S (constants unless the caller seeds derivative slots)
template <class S>
inline std::vector<S> table_as(const Params& p) {
  std::vector<S> t((size_t)(p.cool_law == 1 && p.tab ? p.ntab : 0));
  for (size_t k = 0; k < t.size(); ++k) t[k] = S(p.tab[k]);
  return t;
}

template <class S>
inline void cool(const S U[5], double dt, const Params& p, const S* tab, S out[5]) {
  S rho = U[0];
  S Ek = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / rho;
  S Eth = U[4] - Ek;
  S Efloor = rho * p.t_floor / (p.gamma - 1.0);
  int mode = p.cool_mode;
  if (mode == 2) {                              // masked choice per cell, reading A26
    S Edot_n = cool_rate(Eth, rho, p, tab);
    mode = (dt * std::fabs(val(Edot_n)) > p.f_sub * std::fabs(val(Eth))) ? 0 : 1;
  }
  if (mode == 1) {                              // Eq. 22
    S Edot_n = cool_rate(Eth, rho, p, tab);
    S Epred = smax(Efloor, S(Eth + Edot_n * dt));
    S Edot_p = cool_rate(Epred, rho, p, tab);
    Eth = smax(Efloor, S(Eth + (0.5 * dt) * (Edot_n + Edot_p)));
  } else {                                      // Eq. 23
    const int nsub = p.cool_nsub > 1 ? p.cool_nsub : 1;
    const double ddt = dt / nsub;
    for (int k = 0; k < nsub; ++k) Eth = smax(Efloor, S(Eth + cool_rate(Eth, rho, p, tab) * ddt));
  }
  out[0] = U[0]; out[1] = U[1]; out[2] = U[2]; out[3] = U[3];
  out[4] = Ek + Eth;
}

// ------------------------------------------------------------------------------------------------
// Grid helpers
// ------------------------------------------------------------------------------------------------
struct Grid {
  int n[3];  // nx, ny, nz
  size_t N() const { return (size_t)n[0] * n[1] * n[2]; }
  size_t idx(int i, int j, int k) const { return ((size_t)k * n[1] + j) * n[0] + i; }
};
inline int wrap(int i, int n) { i %= n; return i < 0 ? i + n : i; }

// neighbour of cell (i,j,k) shifted by s cells along axis ax (periodic)
inline size_t shifted(const Grid& g, int i, int j, int k, int ax, int s) {
  int c[3] = {i, j, k};
  c[ax] = wrap(c[ax] + s, g.n[ax]);
  return g.idx(c[0], c[1], c[2]);
}

template <class S>
void compute_prims(const Grid& g, const Params& p, const S* U, S* W) {
  const size_t N = g.N();
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < (long long)N; ++c) {
    S u[5], w[5];
    for (int f = 0; f < 5; ++f) u[f] = U[f * N + c];
    prim(u, p, w);
    for (int f = 0; f < 5; ++f) W[f * N + c] = w[f];
  }
}

// ------------------------------------------------------------------------------------------------
// Step 4 — D(U)_i = sum_a (F_{a,i+1/2} - F_{a,i-1/2}) / dx_a      (Eq. A4, PAPER.md:849;
// roll direction: reading A5).  Natural loop nest with a face-flux array per axis.
// ------------------------------------------------------------------------------------------------
template <class S>
void flux_divergence(const Grid& g, const Params& p, const S* U, S* D) {
  const size_t N = g.N();
  std::vector<S> W(5 * N), F(5 * N);
  compute_prims(g, p, U, W.data());
  for (size_t c = 0; c < 5 * N; ++c) D[c] = S(0.0);
  for (int ax = 0; ax < 3; ++ax) {
    // F[.][cell i] holds the flux through the face i+1/2 along ax
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int i = 0; i < g.n[0]; ++i) {
          size_t cm1 = shifted(g, i, j, k, ax, -1), c0 = g.idx(i, j, k);
          size_t cp1 = shifted(g, i, j, k, ax, +1), cp2 = shifted(g, i, j, k, ax, +2);
          S a[5], b[5], c[5], d[5], f[5];
          for (int q = 0; q < 5; ++q) { a[q] = W[q * N + cm1]; b[q] = W[q * N + c0]; c[q] = W[q * N + cp1]; d[q] = W[q * N + cp2]; }
          face_flux(a, b, c, d, ax, p, f);
          for (int q = 0; q < 5; ++q) F[q * N + c0] = f[q];
        }
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int i = 0; i < g.n[0]; ++i) {
          size_t c0 = g.idx(i, j, k), cm1 = shifted(g, i, j, k, ax, -1);
          for (int q = 0; q < 5; ++q) D[q * N + c0] = D[q * N + c0] + (F[q * N + c0] - F[q * N + cm1]) / p.dx[ax];
        }
  }
}

template <class S>
void apply_cooling(const Grid& g, const Params& p, double dt, S* U) {
  const size_t N = g.N();
  const std::vector<S> tab = table_as<S>(p);
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < (long long)N; ++c) {
    S u[5], o[5];
    for (int f = 0; f < 5; ++f) u[f] = U[f * N + c];
    cool(u, dt, p, tab.data(), o);
    U[4 * N + c] = o[4];
  }
}

// ------------------------------------------------------------------------------------------------
// Step 5 — one full time step.
// integrator 0 (default, reading A1/A2): U* = U^n - dt/2 D(U^n);  U^{n+1} = U^n - dt D(U*)
//                                        (Eqs. A6-A7 form, applied unsplit, Eq. A4)
// integrator 1: Heun RK2: U1 = U^n - dt D(U^n);  U^{n+1} = (U^n + U1 - dt D(U1)) / 2
// integrator 2: SSPRK3 (the paper names the scheme, the stages are the Shu-Osher form):
//               U1 = U^n - dt D(U^n);  U2 = 3/4 U^n + 1/4 (U1 - dt D(U1));  U^{n+1} = 1/3 U^n + 2/3 (U2 - dt D(U2))
// then cooling once (reading A8).
// ------------------------------------------------------------------------------------------------
template <class S>
void step(const Grid& g, const Params& p, const S* U, double dt, S* Uout) {
  const size_t M = 5 * g.N();
  std::vector<S> D(M), Us(M);
  flux_divergence(g, p, U, D.data());
  if (p.integrator == 0) {
    for (size_t c = 0; c < M; ++c) Us[c] = U[c] - (0.5 * dt) * D[c];
    flux_divergence(g, p, Us.data(), D.data());
    for (size_t c = 0; c < M; ++c) Uout[c] = U[c] - dt * D[c];
  } else if (p.integrator == 1) {
    for (size_t c = 0; c < M; ++c) Us[c] = U[c] - dt * D[c];
    flux_divergence(g, p, Us.data(), D.data());
    for (size_t c = 0; c < M; ++c) Uout[c] = 0.5 * (U[c] + (Us[c] - dt * D[c]));
  } else {
    std::vector<S> U2(M);
    for (size_t c = 0; c < M; ++c) Us[c] = U[c] - dt * D[c];
    flux_divergence(g, p, Us.data(), D.data());
    for (size_t c = 0; c < M; ++c) U2[c] = 0.75 * U[c] + 0.25 * (Us[c] - dt * D[c]);
    flux_divergence(g, p, U2.data(), D.data());
    for (size_t c = 0; c < M; ++c) Uout[c] = (1.0 / 3.0) * U[c] + (2.0 / 3.0) * (U2[c] - dt * D[c]);
  }
  if (p.cooling) apply_cooling(g, p, dt, Uout);
}

// ------------------------------------------------------------------------------------------------
// Reverse mode, scatter form (SURVEY.md §8(c) "VJP", dt held constant:
// PAPER.md:876, reading A12).
//
// One stage V = B - tau D(U) with cotangent g on V.  This routine ADDS  -tau J_D(U)^T g  to Ubar.
// Per axis and face i+1/2 the flux cotangent is lambda = (tau/dx_a)(g_{i+1} - g_i); the local
// 5x20 Jacobian of face_flux w.r.t. (W_{i-1}, W_i, W_{i+1}, W_{i+2}) is obtained exactly (to
// rounding) with 20-slot dual numbers through the same face_flux as the forward pass, and its
// transpose times lambda is scattered into Wbar of those four cells.  Finally
// Ubar_i += (dW/dU)_i^T Wbar_i with 5-slot duals through prim().
// ------------------------------------------------------------------------------------------------
inline void stage_vjp_accumulate(const Grid& g, const Params& p, const double* U, double tau,
                                 const double* gV, double* Ubar) {
  const size_t N = g.N();
  std::vector<double> W(5 * N), Wbar(5 * N, 0.0);
  compute_prims(g, p, U, W.data());
  for (int ax = 0; ax < 3; ++ax) {
    // rows along `ax` are independent of each other: parallelise over an outer index that is
    // not the scatter direction
    const int o1 = (ax == 2) ? 1 : 2;  // outer loop axis
    const int o2 = (ax == 0) ? 1 : 0;  // middle loop axis (the remaining one)
#pragma omp parallel for schedule(static)
    for (int a = 0; a < g.n[o1]; ++a)
      for (int b = 0; b < g.n[o2]; ++b)
        for (int s = 0; s < g.n[ax]; ++s) {
          int c[3];
          c[o1] = a; c[o2] = b; c[ax] = s;
          const int i = c[0], j = c[1], k = c[2];
          size_t cell[4] = {shifted(g, i, j, k, ax, -1), g.idx(i, j, k), shifted(g, i, j, k, ax, +1),
                            shifted(g, i, j, k, ax, +2)};
          double lam[5];
          for (int q = 0; q < 5; ++q) lam[q] = (tau / p.dx[ax]) * (gV[q * N + cell[2]] - gV[q * N + cell[1]]);
          Dual<20> w[4][5], f[5];
          for (int m = 0; m < 4; ++m)
            for (int q = 0; q < 5; ++q) { w[m][q] = Dual<20>(W[q * N + cell[m]]); w[m][q].d[m * 5 + q] = 1.0; }
          face_flux(w[0], w[1], w[2], w[3], ax, p, f);
          for (int m = 0; m < 4; ++m)
            for (int q = 0; q < 5; ++q) {
              double acc = 0.0;
              for (int r = 0; r < 5; ++r) acc += f[r].d[m * 5 + q] * lam[r];
              Wbar[q * N + cell[m]] += acc;
            }
        }
  }
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < (long long)N; ++c) {
    Dual<5> u[5], w[5];
    for (int q = 0; q < 5; ++q) { u[q] = Dual<5>(U[q * N + c]); u[q].d[q] = 1.0; }
    prim(u, p, w);
    for (int q = 0; q < 5; ++q) {
      double acc = 0.0;
      for (int r = 0; r < 5; ++r) acc += w[r].d[q] * Wbar[r * N + c];
      Ubar[q * N + c] += acc;
    }
  }
}

// cotangent through the cooling update at U1 (the pre-cooling state): gbar = J_cool(U1)^T g
inline void cooling_vjp(const Grid& g, const Params& p, double dt, const double* U1, const double* gout,
                        double* gbar) {
  const size_t N = g.N();
  const std::vector<Dual<5>> tab = table_as<Dual<5>>(p);
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < (long long)N; ++c) {
    Dual<5> u[5], o[5];
    for (int q = 0; q < 5; ++q) { u[q] = Dual<5>(U1[q * N + c]); u[q].d[q] = 1.0; }
    cool(u, dt, p, tab.data(), o);
    for (int q = 0; q < 5; ++q) {
      double acc = 0.0;
      for (int r = 0; r < 5; ++r) acc += o[r].d[q] * gout[r * N + c];
      gbar[q * N + c] = acc;
    }
  }
}

// VJP of the full step: g_in = (dU^{n+1}/dU^n)^T g_out.
inline void step_vjp(const Grid& g, const Params& p, const double* U, double dt, const double* gout,
                     double* gin) {
  const size_t M = 5 * g.N();
  std::vector<double> D(M), Us(M), g1(M), gs(M, 0.0);
  flux_divergence(g, p, U, D.data());
  if (p.integrator == 0) {
    for (size_t c = 0; c < M; ++c) Us[c] = U[c] - (0.5 * dt) * D[c];
    if (p.cooling) {
      std::vector<double> U1(M);
      flux_divergence(g, p, Us.data(), D.data());
      for (size_t c = 0; c < M; ++c) U1[c] = U[c] - dt * D[c];
      cooling_vjp(g, p, dt, U1.data(), gout, g1.data());
    } else {
      for (size_t c = 0; c < M; ++c) g1[c] = gout[c];
    }
    // U1 = U - dt D(U*):  Ubar += g1,  U*bar += -dt J_D(U*)^T g1
    stage_vjp_accumulate(g, p, Us.data(), dt, g1.data(), gs.data());
    // U* = U - dt/2 D(U):  Ubar += U*bar - dt/2 J_D(U)^T U*bar
    for (size_t c = 0; c < M; ++c) gin[c] = g1[c] + gs[c];
    stage_vjp_accumulate(g, p, U, 0.5 * dt, gs.data(), gin);
  } else if (p.integrator == 2) {
    // SSPRK3: Ua = U - dt D(U); Ub = 3/4 U + 1/4 (Ua - dt D(Ua)); U1 = 1/3 U + 2/3 (Ub - dt D(Ub))
    std::vector<double> Ub(M), Da(M);
    for (size_t c = 0; c < M; ++c) Us[c] = U[c] - dt * D[c];
    flux_divergence(g, p, Us.data(), Da.data());
    for (size_t c = 0; c < M; ++c) Ub[c] = 0.75 * U[c] + 0.25 * (Us[c] - dt * Da[c]);
    if (p.cooling) {
      std::vector<double> U1(M);
      flux_divergence(g, p, Ub.data(), D.data());
      for (size_t c = 0; c < M; ++c) U1[c] = (1.0 / 3.0) * U[c] + (2.0 / 3.0) * (Ub[c] - dt * D[c]);
      cooling_vjp(g, p, dt, U1.data(), gout, g1.data());
    } else {
      for (size_t c = 0; c < M; ++c) g1[c] = gout[c];
    }
    std::vector<double> a(M), b(M), gb(M), ga(M);
    for (size_t c = 0; c < M; ++c) { a[c] = (2.0 / 3.0) * g1[c]; gb[c] = a[c]; }   // Ubbar = 2/3 g1 ...
    stage_vjp_accumulate(g, p, Ub.data(), dt, a.data(), gb.data());                // ... - dt J_D(Ub)^T (2/3 g1)
    for (size_t c = 0; c < M; ++c) { b[c] = 0.25 * gb[c]; ga[c] = b[c]; }          // Uabar = 1/4 Ubbar ...
    stage_vjp_accumulate(g, p, Us.data(), dt, b.data(), ga.data());                // ... - dt J_D(Ua)^T (1/4 Ubbar)
    for (size_t c = 0; c < M; ++c) gin[c] = (1.0 / 3.0) * g1[c] + 0.75 * gb[c] + ga[c];
    stage_vjp_accumulate(g, p, U, dt, ga.data(), gin);                             // ... - dt J_D(U)^T Uabar
  } else {
    // Heun: Ua = U - dt D(U); U1 = (U + Ua - dt D(Ua)) / 2
    for (size_t c = 0; c < M; ++c) Us[c] = U[c] - dt * D[c];
    if (p.cooling) {
      std::vector<double> U1(M);
      flux_divergence(g, p, Us.data(), D.data());
      for (size_t c = 0; c < M; ++c) U1[c] = 0.5 * (U[c] + (Us[c] - dt * D[c]));
      cooling_vjp(g, p, dt, U1.data(), gout, g1.data());
    } else {
      for (size_t c = 0; c < M; ++c) g1[c] = gout[c];
    }
    std::vector<double> h(M);
    for (size_t c = 0; c < M; ++c) { h[c] = 0.5 * g1[c]; gs[c] = h[c]; }   // Uabar = g1/2 + ...
    stage_vjp_accumulate(g, p, Us.data(), dt, h.data(), gs.data());       // ... - dt J_D(Ua)^T g1/2
    for (size_t c = 0; c < M; ++c) gin[c] = h[c] + gs[c];                  // Ubar = g1/2 + Uabar ...
    stage_vjp_accumulate(g, p, U, dt, gs.data(), gin);                     // ... - dt J_D(U)^T Uabar
  }
}

// ------------------------------------------------------------------------------------------------
// CFL time step, Eq. A8:  dt = C min_a dx_a / max_cells(|v_a| + c_s).
// The "dt recipe" of SURVEY.md §8(c): every operation in T, in exactly this order, no FMA
// contraction (this file is compiled with -ffp-contract=off), constants formed in double and
// rounded to T once.  Returns 0, or -4 if any input or wave speed is not finite.
// ------------------------------------------------------------------------------------------------
template <class T>
int cfl_dt(const Grid& g, const Params& p, double cfl, const T* U, double* dt_out, double smax_out[3]) {
  const size_t N = g.N();
  const T gam = (T)p.gamma, gm1 = (T)(p.gamma - 1.0);
  const T rfl = (T)p.rho_floor, pfl = (T)p.p_floor, half = (T)0.5;
  T Smax[3] = {(T)0, (T)0, (T)0};
  T S0 = (T)0, S1 = (T)0, S2 = (T)0;
  int nbad = 0;
  // max is exact and order-independent, so the thread count cannot change a bit of the result
#pragma omp parallel for schedule(static) reduction(max : S0, S1, S2) reduction(+ : nbad)
  for (long long c = 0; c < (long long)N; ++c) {
    T rho = U[c], mx = U[N + c], my = U[2 * N + c], mz = U[3 * N + c], E = U[4 * N + c];
    T rt = (rho >= rfl) ? rho : rfl;
    T vx = mx / rt, vy = my / rt, vz = mz / rt;
    T q = ((mx * mx) + (my * my)) + (mz * mz);
    T P = gm1 * (E - half * (q / rt));
    P = (P >= pfl) ? P : pfl;
    T cs = std::sqrt((gam * P) / rt);
    T sx = std::fabs(vx) + cs, sy = std::fabs(vy) + cs, sz = std::fabs(vz) + cs;
    // the floors (a compare-select) would silently swallow a NaN in rho or E: test the inputs too
    if (!std::isfinite(rho) || !std::isfinite(mx) || !std::isfinite(my) || !std::isfinite(mz) || !std::isfinite(E) ||
        !std::isfinite(sx) || !std::isfinite(sy) || !std::isfinite(sz)) nbad += 1;
    if (sx > S0) S0 = sx;
    if (sy > S1) S1 = sy;
    if (sz > S2) S2 = sz;
  }
  Smax[0] = S0; Smax[1] = S1; Smax[2] = S2;
  for (int a = 0; a < 3; ++a) smax_out[a] = (double)Smax[a];
  if (nbad) return -4;
  T best = (T)0;
  bool first = true;
  for (int a = 0; a < 3; ++a) {
    T dxa = (T)p.dx[a];
    T r = dxa / Smax[a];
    if (first || r < best) { best = r; first = false; }
  }
  T dt = (T)cfl * best;
  *dt_out = (double)dt;
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Cooling-time limit on the time step, Eqs. 20-21.
//   t_cool(x) = |E_th| / |n_H Gamma - n_H^2 Lambda|                                          (Eq. 20)
//   dt <= min(dt_hydro, c_cool min_x t_cool(x), dt_max)                                       (Eq. 21)
// Code units of this file (reading A10): n_H = rho, Gamma = 0, Lambda = lambda0 T^alpha, T = (gamma-1) E_th / rho,
// so the denominator is |Edot| of cool_rate().  Reading A24: E_th is taken from the conserved variables exactly as
// cool() does (no floors); the per-cell quotient is formed in double whatever the array type (the power function has
// no bit-exact definition to share, unlike the recipe of Eq. A8); a cell with zero rate (T <= 0) has t_cool = +inf
// and never decides the minimum; cells already on the temperature floor are NOT exempted (the paper exempts none).
// The three candidates of Eq. 21 are compared in T: dt = min(dt_hydro, T(c_cool * tmin), T(dt_max)); c_cool <= 0
// or dt_max <= 0 switches that candidate off.
// ------------------------------------------------------------------------------------------------
inline double t_cool_cell(const double U[5], const Params& p) {
  double rho = U[0];
  double Ek = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / rho;
  double Eth = U[4] - Ek;
  double Edot = cool_rate<double>(Eth, rho, p, p.tab);
  if (Edot == 0.0) return std::numeric_limits<double>::infinity();
  return std::fabs(Eth) / std::fabs(Edot);
}

template <class T>
double t_cool_min(const Grid& g, const Params& p, const T* U) {
  const size_t N = g.N();
  double best = std::numeric_limits<double>::infinity();
  for (size_t c = 0; c < N; ++c) {
    double u[5];
    for (int f = 0; f < 5; ++f) u[f] = (double)U[f * N + c];
    double t = t_cool_cell(u, p);
    if (t < best) best = t;
  }
  return best;
}

template <class T>
double limited_dt(double dt_hydro, double tmin, double c_cool, double dt_max) {
  T dt = (T)dt_hydro;
  if (c_cool > 0.0) { T dc = (T)(c_cool * tmin); if (dc < dt) dt = dc; }
  if (dt_max > 0.0) { T dm = (T)dt_max; if (dm < dt) dt = dm; }
  return (double)dt;
}

// ------------------------------------------------------------------------------------------------
// Decision margins (test infrastructure for the VJP parity check; "non-smooth operators",
// PAPER.md:119-127; readings A7 / A17).
//
// The scheme is piecewise smooth: its a.e. derivative follows the branch actually taken by every compare the step
// makes — limiter (a b <= 0, |a| <= |b|), Eq. A3's min / max, the HLLC / HLL select order (S_L >= 0, S_R <= 0,
// S* >= 0), Rusanov's max of absolute values, the floors of prim().  An implementation that evaluates the same
// formulas in another precision takes the same branch unless the two compared quantities agree to within its
// rounding error.  For every compare this routine returns how far the oracle's own operands are from the tie,
// divided by the magnitude on which rounding errors of those operands scale:
//   rho: rho;   velocities: |v| + c_s;   pressure: P + (gamma-1) rho |v|^2 / 2  (P is a difference of E and E_kin)
// (the largest of these over the cells the operands are formed from).  Output M[4][N]:
//   M[a][i], a = 0..2: min over the five limiter calls at cell i along axis a and the Riemann compares at face i+1/2
//   M[3][i]: the two floors of prim() at cell i.
// A compare whose operands are exactly equal because the data are exactly uniform there (a = b = 0) is not a tie in
// this sense: identical inputs give identical operands in any deterministic arithmetic; it gets +inf.
// ------------------------------------------------------------------------------------------------
inline void margin_scales(const double W[5], double gamma, double s[5]) {
  const double vv = std::sqrt(W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
  const double cs = std::sqrt(gamma * W[4] / W[0]);
  s[0] = W[0];
  s[1] = s[2] = s[3] = vv + cs;
  s[4] = W[4] + 0.5 * (gamma - 1.0) * W[0] * vv * vv;
}

inline double limiter_margin(double a, double b, int kind, double s) {
  const double inf = std::numeric_limits<double>::infinity();
  if (kind == 3) return inf;
  if (a == 0.0 && b == 0.0) return inf;
  const double fa = std::fabs(a), fb = std::fabs(b);
  double m = (fa < fb ? fa : fb) / s;                       // a b <= 0 flips when either operand crosses zero
  if (a * b <= 0.0) return m;
  if (kind == 0) {                                          // minmod: |a| <= |b|
    m = std::fmin(m, std::fabs(fa - fb) / s);
  } else if (kind == 2) {                                   // MC: |2a| <= |2b|, then |m| <= |(a+b)/2|
    m = std::fmin(m, 2.0 * std::fabs(fa - fb) / s);
    m = std::fmin(m, std::fabs(2.0 * (fa < fb ? fa : fb) - 0.5 * (fa + fb)) / s);
  }
  return m;                                                 // van Leer: smooth away from a b = 0
}

// the compares riemann() makes on the face states L, R (same expressions as riemann() above)
inline double riemann_margin(const double L[5], const double R[5], int ax, const Params& p) {
  const double inf = std::numeric_limits<double>::infinity();
  const double g = p.gamma;
  const double uL = L[1 + ax], uR = R[1 + ax];
  const double cL = std::sqrt(g * L[4] / L[0]), cR = std::sqrt(g * R[4] / R[0]);
  const double s = std::fmax(std::fabs(uL) + cL, std::fabs(uR) + cR);
  // L and R agree in (rho, u_n, P) to rounding: either the data are uniform there, or both cells' limiters returned the
  // difference they share, so that L = W_i + d/2 and R = W_{i+1} - d/2 are the same function of the data; whichever
  // argument Eq. A3's min / max then return, the derivative with respect to the data is the same: not a tie
  const double rs[3] = {std::fmax(L[0], R[0]), s, std::fmax(L[4], R[4])};
  const int qs[3] = {0, 1 + ax, 4};
  bool same = true;
  for (int m3 = 0; m3 < 3; ++m3) same = same && (std::fabs(L[qs[m3]] - R[qs[m3]]) <= 1e-14 * rs[m3]);
  const double SL = std::fmin(uL - cL, uR - cR), SR = std::fmax(uL + cL, uR + cR);
  double m = inf;
  if (!same) {                                              // which argument Eq. A3's min / max return
    m = std::fmin(m, std::fabs((uL - cL) - (uR - cR)) / s);
    m = std::fmin(m, std::fabs((uL + cL) - (uR + cR)) / s);
  }
  if (p.riemann == 2) {                                     // max(|S_L|, |S_R|) and the two absolute values
    m = std::fmin(m, std::fabs(std::fabs(SL) - std::fabs(SR)) / s);
    m = std::fmin(m, std::fabs(SL) / s);
    m = std::fmin(m, std::fabs(SR) / s);
    return m;
  }
  m = std::fmin(m, std::fabs(SL) / s);                      // S_L >= 0
  m = std::fmin(m, std::fabs(SR) / s);                      // S_R <= 0
  if (p.riemann == 0 && SL < 0.0 && SR > 0.0) {             // S* >= 0
    const double Ss = (R[4] - L[4] + L[0] * uL * (SL - uL) - R[0] * uR * (SR - uR)) /
                      (L[0] * (SL - uL) - R[0] * (SR - uR));
    m = std::fmin(m, std::fabs(Ss) / s);
  }
  return m;
}

inline void decision_margins(const Grid& g, const Params& p, const double* U, double* M) {
  const size_t N = g.N();
  std::vector<double> W(5 * N), Sc(5 * N);
  compute_prims(g, p, U, W.data());
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < (long long)N; ++c) {
    double w[5], s[5];
    for (int q = 0; q < 5; ++q) w[q] = W[q * N + c];
    margin_scales(w, p.gamma, s);
    for (int q = 0; q < 5; ++q) Sc[q * N + c] = s[q];
    // floors of prim(): rho >= rho_floor, P >= p_floor, on the unfloored values
    const double rho = U[c];
    const double rr = std::fmax(rho, p.rho_floor);
    const double Praw = (p.gamma - 1.0) * (U[4 * N + c] - 0.5 * (U[N + c] * U[N + c] + U[2 * N + c] * U[2 * N + c] + U[3 * N + c] * U[3 * N + c]) / rr);
    const double sP = std::fabs(Praw) + 0.5 * (p.gamma - 1.0) * (U[N + c] * U[N + c] + U[2 * N + c] * U[2 * N + c] + U[3 * N + c] * U[3 * N + c]) / rr;
    M[3 * N + c] = std::fmin(std::fabs(rho - p.rho_floor) / std::fmax(std::fabs(rho), p.rho_floor),
                             std::fabs(Praw - p.p_floor) / std::fmax(sP, p.p_floor));
  }
  for (int ax = 0; ax < 3; ++ax) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int i = 0; i < g.n[0]; ++i) {
          const size_t cm1 = shifted(g, i, j, k, ax, -1), c0 = g.idx(i, j, k);
          const size_t cp1 = shifted(g, i, j, k, ax, +1), cp2 = shifted(g, i, j, k, ax, +2);
          double a[5], b[5], c[5], d[5], WL[5], WR[5];
          for (int q = 0; q < 5; ++q) { a[q] = W[q * N + cm1]; b[q] = W[q * N + c0]; c[q] = W[q * N + cp1]; d[q] = W[q * N + cp2]; }
          double m = std::numeric_limits<double>::infinity();
          for (int q = 0; q < 5; ++q) {                     // the limiter call of cell i (Eq. A1)
            const double s = std::fmax(Sc[q * N + cm1], std::fmax(Sc[q * N + c0], Sc[q * N + cp1]));
            m = std::fmin(m, limiter_margin(c[q] - b[q], b[q] - a[q], p.limiter, s));
          }
          face_states(a, b, c, d, p, WL, WR);
          m = std::fmin(m, riemann_margin(WL, WR, ax, p));
          M[(size_t)ax * N + c0] = m;
        }
  }
}

// Conditioning of the limiter's derivative (van Leer only): d lim / da = 2 b^2 / (a + b)^2 is smooth but depends on the RATIO of the
// two differences: an error eps s in them (s: the rounding scale of margin_scales) changes it by at most ~ 12 eps s / (|a| + |b|)
// (|d/da|, |d/db| of 2 b^2 / (a+b)^2 are bounded by 4 / (a + b) for a b > 0).
// C[a][i] = max over the five fields of s / (|a| + |b|) at cell i along axis a where the slope is active (a b > 0), else 0.
// minmod and MC have piecewise-constant derivatives: C = 0.
inline void limiter_conditioning(const Grid& g, const Params& p, const double* U, double* C) {
  const size_t N = g.N();
  std::vector<double> W(5 * N);
  compute_prims(g, p, U, W.data());
  for (int ax = 0; ax < 3; ++ax) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
      for (int j = 0; j < g.n[1]; ++j)
        for (int i = 0; i < g.n[0]; ++i) {
          const size_t cm1 = shifted(g, i, j, k, ax, -1), c0 = g.idx(i, j, k), cp1 = shifted(g, i, j, k, ax, +1);
          double worst = 0.0;
          if (p.limiter == 1) {
            double w[3][5], sc[3][5];
            const size_t cs[3] = {cm1, c0, cp1};
            for (int m = 0; m < 3; ++m) {
              for (int q = 0; q < 5; ++q) w[m][q] = W[q * N + cs[m]];
              margin_scales(w[m], p.gamma, sc[m]);
            }
            for (int q = 0; q < 5; ++q) {
              const double a = w[2][q] - w[1][q], b = w[1][q] - w[0][q];
              if (a * b <= 0.0) continue;
              const double s = std::fmax(sc[0][q], std::fmax(sc[1][q], sc[2][q]));
              worst = std::fmax(worst, s / (std::fabs(a) + std::fabs(b)));
            }
          }
          C[(size_t)ax * N + c0] = worst;
        }
  }
}

// the compares of cool() at the pre-cooling state U1: T > 0 and (law 1) T < t_switch and the table interval inside every
// cool_rate(), every max with E_floor, and (mode 2) the masked choice of the integrator; relative to E_kin + |E_th| (E_th is
// a difference of E and E_kin)
inline double rate_margin(double Eth, double rho, double s, const Params& p) {
  double m = std::fabs(Eth) / s;                                               // T > 0
  if (p.cool_law == 1) {
    const double Esw = rho * p.t_switch / (p.gamma - 1.0);
    m = std::fmin(m, std::fabs(Eth - Esw) / s);                                // T < t_switch
    const double T = (p.gamma - 1.0) * Eth / rho;
    if (T >= p.t_switch) {                                                     // kinks of the interpolant at the nodes
      const double u = (std::log10(T) - p.tab_logT0) / p.tab_dlogT;
      if (u > 0.0 && u < (double)(p.ntab - 1)) {
        const double fr = u - std::floor(u);
        m = std::fmin(m, 2.302585092994045684 * p.tab_dlogT * std::fmin(fr, 1.0 - fr) * std::fabs(Eth) / s);
      }
    }
  }
  return m;
}

inline void cooling_margins(const Grid& g, const Params& p, double dt, const double* U1, double* M) {
  const size_t N = g.N();
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < (long long)N; ++c) {
    const double rho = U1[c];
    const double Ek = 0.5 * (U1[N + c] * U1[N + c] + U1[2 * N + c] * U1[2 * N + c] + U1[3 * N + c] * U1[3 * N + c]) / rho;
    double Eth = U1[4 * N + c] - Ek;
    const double s = Ek + std::fabs(Eth);
    const double Efloor = rho * p.t_floor / (p.gamma - 1.0);
    double m = rate_margin(Eth, rho, s, p);
    int mode = p.cool_mode;
    if (mode == 2) {
      const double En = cool_rate<double>(Eth, rho, p, p.tab);
      m = std::fmin(m, std::fabs(dt * std::fabs(En) - p.f_sub * std::fabs(Eth)) / (p.f_sub * s));
      mode = (dt * std::fabs(En) > p.f_sub * std::fabs(Eth)) ? 0 : 1;
    }
    if (mode == 1) {
      const double En = cool_rate<double>(Eth, rho, p, p.tab);
      const double raw = Eth + En * dt;
      m = std::fmin(m, std::fabs(raw - Efloor) / s);
      const double Epred = std::fmax(Efloor, raw);
      m = std::fmin(m, rate_margin(Epred, rho, s, p));
      const double raw2 = Eth + (0.5 * dt) * (En + cool_rate<double>(Epred, rho, p, p.tab));
      m = std::fmin(m, std::fabs(raw2 - Efloor) / s);
    } else {
      const int nsub = p.cool_nsub > 1 ? p.cool_nsub : 1;
      const double ddt = dt / nsub;
      for (int k = 0; k < nsub; ++k) {
        if (k > 0) m = std::fmin(m, rate_margin(Eth, rho, s, p));
        const double raw = Eth + cool_rate<double>(Eth, rho, p, p.tab) * ddt;
        m = std::fmin(m, std::fabs(raw - Efloor) / s);
        Eth = std::fmax(Efloor, raw);
      }
    }
    M[c] = m;
  }
}

// ------------------------------------------------------------------------------------------------
// Gradient with respect to the cooling table itself ("... and even the cooling tables themselves"):
//   gtab[k] = sum_cells gout_E(cell) * d E_out(cell) / d tab[k]     at the pre-cooling state U1,
// by dual numbers with one derivative slot per table node through the same cool() (ntab <= 32).
// ------------------------------------------------------------------------------------------------
inline int cooling_table_vjp(const Grid& g, const Params& p, double dt, const double* U1, const double* gout, double* gtab) {
  constexpr int NT = 32;
  if (p.cool_law != 1 || !p.tab || p.ntab > NT) return -1;
  const size_t N = g.N();
  std::vector<Dual<NT>> tab((size_t)p.ntab);
  for (int k = 0; k < p.ntab; ++k) { tab[k] = Dual<NT>(p.tab[k]); tab[k].d[k] = 1.0; }
  for (int k = 0; k < p.ntab; ++k) gtab[k] = 0.0;
  for (size_t c = 0; c < N; ++c) {                 // plain serial sum: a fixed order
    Dual<NT> u[5], o[5];
    for (int q = 0; q < 5; ++q) u[q] = Dual<NT>(U1[q * N + c]);
    cool(u, dt, p, tab.data(), o);
    for (int k = 0; k < p.ntab; ++k) gtab[k] += o[4].d[k] * gout[4 * N + c];
  }
  return 0;
}

}  // namespace dho
