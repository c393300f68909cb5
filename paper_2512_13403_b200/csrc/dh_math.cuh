// dh_math.cuh — pointwise device arithmetic of the Euler finite-volume step (sm_100a).
//
// Primitive conversion (Eq. 2), limited slopes (Eq. A1), the HLLC flux with
// the wave-speed estimates of Eq. A3, the HLL and Rusanov alternatives, the cooling update (Eq. 23) and the
// hand-written reverse-mode counterparts of each.  The formulas are arranged for instruction count
// (one reciprocal per density, star state evaluated on the upwind side only, transverse momentum flux
// as v_t * F_mass, the supersonic branches folded into S_eff = min(S_L,0) / max(S_R,0)); they are
// algebraically the textbook HLLC and agree with the CPU oracle to rounding.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace dh {

// ------------------------------------------------------------------------------------------------
// scalar helpers: fp32 uses the MUFU approximations (rel. error ~1e-7, far inside the 2e-5 bar),
// fp64 uses IEEE division / sqrt.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float rcp_(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
__device__ __forceinline__ float sqrt_(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
__device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double min_(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double max_(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float abs_(float a) { return fabsf(a); }
__device__ __forceinline__ double abs_(double a) { return fabs(a); }
__device__ __forceinline__ float pow_(float a, float b) { return __powf(a, b); }
__device__ __forceinline__ double pow_(double a, double b) { return pow(a, b); }

template <class T>
struct Consts {
  T gamma;      // adiabatic index
  T gm1;        // gamma - 1
  T inv_gm1;    // 1 / (gamma - 1)
  T rho_floor, p_floor;
  // cooling
  T lambda0, alpha, t_floor;
  int alpha_is_half;
  int cool_mode, cool_nsub;   // DH_OPT_COOL_MODE / DH_OPT_COOL_NSUB; (0, 1) is the update fused into the stage kernels
  // two-branch law of Eqs. 17-19 (DH_OPT_COOL_LAW = 1): Koyama-Inutsuka fit + uniform heating below
  // t_switch, tabulated Lambda_CIE above it.  The table holds log2 Lambda at nodes equally spaced in log2 T (the same
  // interpolant as in log10-log10: a change of base is linear), so that one lg2 / ex2 pair evaluates it.
  int cool_law;
  T t_switch, lambda1, alpha1, lambda2, alpha2, gamma0;
  T f_sub;                    // DH_OPT_COOL_FSUB: cool_mode 2 sub-cycles a cell when dt |Edot| > f_sub |E_th| (reading A26)
  const T* tab;               // DEVICE, ntab values of log2 Lambda
  int ntab;
  T tab_l2t0, tab_inv_dl2t;   // first node and 1 / spacing, in log2 T
};

__device__ __forceinline__ float log2_(float x) { return __log2f(x); }
__device__ __forceinline__ double log2_(double x) { return log2(x); }
__device__ __forceinline__ float exp2_(float x) { return exp2f(x); }
__device__ __forceinline__ double exp2_(double x) { return exp2(x); }
__device__ __forceinline__ float floor_(float x) { return floorf(x); }
__device__ __forceinline__ double floor_(double x) { return floor(x); }

// ------------------------------------------------------------------------------------------------
// primitives  W = (rho, vx, vy, vz, P); floors act only here (reading A6)
// ------------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ void prim(const T U[5], const Consts<T>& c, T W[5]) {
  T rho = max_(U[0], c.rho_floor);
  T r = rcp_(rho);
  T vx = U[1] * r, vy = U[2] * r, vz = U[3] * r;
  T ke = T(0.5) * (U[1] * vx + U[2] * vy + U[3] * vz);
  W[0] = rho; W[1] = vx; W[2] = vy; W[3] = vz;
  W[4] = max_(c.gm1 * (U[4] - ke), c.p_floor);
}

// Ubar += (dW/dU)^T Wbar   (floor masks: derivative 0 where floored)
template <class T>
__device__ __forceinline__ void prim_vjp(const T U[5], const Consts<T>& c, const T Wb[5], T Ub[5]) {
  T rho = max_(U[0], c.rho_floor);
  T r = rcp_(rho);
  T vx = U[1] * r, vy = U[2] * r, vz = U[3] * r;
  T ke = T(0.5) * (U[1] * vx + U[2] * vy + U[3] * vz);
  T Pb = (c.gm1 * (U[4] - ke) >= c.p_floor) ? Wb[4] : T(0);
  T gP = c.gm1 * Pb;
  Ub[4] = gP;
  Ub[1] = Wb[1] * r - gP * vx;
  Ub[2] = Wb[2] * r - gP * vy;
  Ub[3] = Wb[3] * r - gP * vz;
  T rb = Wb[0] - (Wb[1] * vx + Wb[2] * vy + Wb[3] * vz) * r + T(0.5) * gP * (vx * vx + vy * vy + vz * vz);
  Ub[0] = (U[0] >= c.rho_floor) ? rb : T(0);
}

// ------------------------------------------------------------------------------------------------
// slope limiters, a = W_{i+1}-W_i, b = W_i-W_{i-1}.  LIM: 0 minmod, 1 van Leer, 2 MC.
// minmod(a,b) = median(a, b, 0): two min/max pairs, no multiply, no branch.
// ------------------------------------------------------------------------------------------------
template <class T, int LIM>
__device__ __forceinline__ T limit(T a, T b) {
  if (LIM == 0) {
    T mn = min_(a, b), mx = max_(a, b);
    return min_(max_(mn, T(0)), mx);
  } else if (LIM == 1) {
    T ab = a * b;
    return (ab > T(0)) ? T(2) * ab * rcp_(a + b) : T(0);
  } else {
    T ab = a * b;
    T mn = min_(a, b), mx = max_(a, b);
    T m2 = T(2) * min_(max_(mn, T(0)), mx);   // 2 minmod(a,b)
    T cc = T(0.5) * (a + b);
    T r = (abs_(m2) <= abs_(cc)) ? m2 : cc;
    return (ab > T(0)) ? r : T(0);
  }
}

// partial derivatives of the limiter on the branch taken (ties: |a| == |b| -> a; a b <= 0 -> 0)
template <class T, int LIM>
__device__ __forceinline__ void limit_grad(T a, T b, T& da, T& db) {
  const bool on = (a * b > T(0));
  if (LIM == 0) {
    const bool pa = abs_(a) <= abs_(b);
    da = (on && pa) ? T(1) : T(0);
    db = (on && !pa) ? T(1) : T(0);
  } else if (LIM == 1) {
    T s = rcp_(a + b);
    T s2 = T(2) * s * s;
    da = on ? s2 * b * b : T(0);
    db = on ? s2 * a * a : T(0);
  } else {
    const bool pa = abs_(a) <= abs_(b);
    T m2 = T(2) * (pa ? a : b);
    T cc = T(0.5) * (a + b);
    const bool pm = abs_(m2) <= abs_(cc);
    da = on ? (pm ? (pa ? T(2) : T(0)) : T(0.5)) : T(0);
    db = on ? (pm ? (pa ? T(0) : T(2)) : T(0.5)) : T(0);
  }
}

// ------------------------------------------------------------------------------------------------
// HLLC flux through a face with normal axis AX from left/right primitive states (rho, vx, vy, vz, P).
// F is in conserved-field order (rho, mx, my, mz, E).
// ------------------------------------------------------------------------------------------------
template <class T, int AX>
__device__ __forceinline__ void hllc(const T L[5], const T R[5], const Consts<T>& c, T F[5]) {
  constexpr int n = 1 + AX, t1 = 1 + (AX + 1) % 3, t2 = 1 + (AX + 2) % 3;
  const T rL = rcp_(L[0]), rR = rcp_(R[0]);
  const T cL = sqrt_(c.gamma * L[4] * rL), cR = sqrt_(c.gamma * R[4] * rR);
  const T uL = L[n], uR = R[n];
  const T SL = min_(uL - cL, uR - cR);          // Eq. A3
  const T SR = max_(uL + cL, uR + cR);
  const T aL = L[0] * (SL - uL), aR = R[0] * (SR - uR);
  const T num = (R[4] - L[4]) + aL * uL - aR * uR;
  const T Ss = num * rcp_(aL - aR);             // contact speed S*
  const bool left = (Ss >= T(0));
  const T rhoK = left ? L[0] : R[0], uK = left ? uL : uR, v1 = left ? L[t1] : R[t1], v2 = left ? L[t2] : R[t2];
  const T PK = left ? L[4] : R[4], SK = left ? SL : SR, aK = left ? aL : aR, rK = left ? rL : rR;
  const T Seff = left ? min_(SK, T(0)) : max_(SK, T(0));   // 0 in the supersonic branches -> F = F_K
  const T e = PK * rK * c.inv_gm1 + T(0.5) * (uK * uK + v1 * v1 + v2 * v2);   // E_K / rho_K
  const T EK = rhoK * e, mK = rhoK * uK;
  const T inv = rcp_(SK - Ss);
  const T fac = aK * inv;                       // rho*_K
  const T Fm = mK + Seff * (fac - rhoK);
  const T Es = inv * (aK * e + (Ss - uK) * (aK * Ss + PK));   // E*_K
  F[0] = Fm;
  F[n] = mK * uK + PK + Seff * (fac * Ss - mK);
  F[t1] = v1 * Fm;
  F[t2] = v2 * Fm;
  F[4] = uK * (EK + PK) + Seff * (Es - EK);
}

// (Lb, Rb) += (dF/dL, dF/dR)^T Fb   — reverse of hllc() above, statement by statement.
template <class T, int AX>
__device__ __forceinline__ void hllc_vjp(const T L[5], const T R[5], const Consts<T>& c, const T Fb[5], T Lb[5], T Rb[5]) {
  constexpr int n = 1 + AX, t1 = 1 + (AX + 1) % 3, t2 = 1 + (AX + 2) % 3;
  // ---- forward recompute
  const T rL = rcp_(L[0]), rR = rcp_(R[0]);
  const T cL = sqrt_(c.gamma * L[4] * rL), cR = sqrt_(c.gamma * R[4] * rR);
  const T uL = L[n], uR = R[n];
  const T sLa = uL - cL, sLb = uR - cR, sRa = uL + cL, sRb = uR + cR;
  const bool pickLa = (sLa <= sLb), pickRa = (sRa >= sRb);
  const T SL = pickLa ? sLa : sLb, SR = pickRa ? sRa : sRb;
  const T dL = SL - uL, dR = SR - uR;
  const T aL = L[0] * dL, aR = R[0] * dR;
  const T num = (R[4] - L[4]) + aL * uL - aR * uR;
  const T iden = rcp_(aL - aR);
  const T Ss = num * iden;
  const bool left = (Ss >= T(0));
  const T rhoK = left ? L[0] : R[0], uK = left ? uL : uR, v1 = left ? L[t1] : R[t1], v2 = left ? L[t2] : R[t2];
  const T PK = left ? L[4] : R[4], SK = left ? SL : SR, aK = left ? aL : aR, rK = left ? rL : rR;
  const bool seff_on = left ? (SK < T(0)) : (SK > T(0));
  const T Seff = seff_on ? SK : T(0);
  const T e = PK * rK * c.inv_gm1 + T(0.5) * (uK * uK + v1 * v1 + v2 * v2);
  const T EK = rhoK * e, mK = rhoK * uK;
  const T inv = rcp_(SK - Ss);
  const T fac = aK * inv;
  const T Fm = mK + Seff * (fac - rhoK);
  const T Y = Ss - uK, Z = aK * Ss + PK;
  const T X = aK * e + Y * Z;
  const T Es = inv * X;
  // ---- reverse
  const T Fmb = Fb[0] + Fb[t1] * v1 + Fb[t2] * v2;    // F_t = v_t * F_m
  T v1b = Fb[t1] * Fm, v2b = Fb[t2] * Fm;
  // F_E = uK (EK + PK) + Seff (Es - EK)
  T uKb = Fb[4] * (EK + PK);
  T EKb = Fb[4] * (uK - Seff);
  T PKb = Fb[4] * uK;
  T Seffb = Fb[4] * (Es - EK);
  const T Esb = Fb[4] * Seff;
  // Es = inv * X,  X = aK e + Y Z
  T invb = Esb * X;
  const T Xb = Esb * inv;
  T aKb = Xb * e;
  T eb = Xb * aK;
  const T Yb = Xb * Z, Zb = Xb * Y;
  T Ssb = Yb;
  uKb -= Yb;
  aKb += Zb * Ss;
  Ssb += Zb * aK;
  PKb += Zb;
  // F_n = mK uK + PK + Seff (fac Ss - mK)
  T mKb = Fb[n] * (uK - Seff);
  uKb += Fb[n] * mK;
  PKb += Fb[n];
  Seffb += Fb[n] * (fac * Ss - mK);
  T facb = Fb[n] * Seff * Ss;
  Ssb += Fb[n] * Seff * fac;
  // F_m = mK + Seff (fac - rhoK)
  mKb += Fmb;
  Seffb += Fmb * (fac - rhoK);
  facb += Fmb * Seff;
  T rhoKb = -Fmb * Seff;
  // fac = aK inv; inv = 1 / (SK - Ss)
  aKb += facb * inv;
  invb += facb * aK;
  const T wb = -invb * inv * inv;
  T SKb = wb;
  Ssb -= wb;
  // mK = rhoK uK; EK = rhoK e; e = PK rK / (gamma-1) + q/2
  rhoKb += mKb * uK;
  uKb += mKb * rhoK;
  rhoKb += EKb * e;
  eb += EKb * rhoK;
  PKb += eb * rK * c.inv_gm1;
  const T rKb = eb * PK * c.inv_gm1;
  uKb += eb * uK;
  v1b += eb * v1;
  v2b += eb * v2;
  // Seff = SK on its active branch
  if (seff_on) SKb += Seffb;
  // un-select K
  T rhoLb = T(0), rhoRb = T(0), uLb = T(0), uRb = T(0), PLb = T(0), PRb = T(0);
  T SLb = T(0), SRb = T(0), aLb = T(0), aRb = T(0), rLb = T(0), rRb = T(0);
  if (left) { rhoLb = rhoKb; uLb = uKb; Lb[t1] += v1b; Lb[t2] += v2b; PLb = PKb; SLb = SKb; aLb = aKb; rLb = rKb; }
  else      { rhoRb = rhoKb; uRb = uKb; Rb[t1] += v1b; Rb[t2] += v2b; PRb = PKb; SRb = SKb; aRb = aKb; rRb = rKb; }
  // Ss = num / den,  den = aL - aR,  num = PR - PL + aL uL - aR uR
  const T numb = Ssb * iden;
  const T denb = -Ssb * Ss * iden;
  aLb += denb + numb * uL;
  aRb -= denb + numb * uR;
  PRb += numb;
  PLb -= numb;
  uLb += numb * aL;
  uRb -= numb * aR;
  // aL = rhoL dL, dL = SL - uL (and R)
  rhoLb += aLb * dL;
  rhoRb += aRb * dR;
  const T dLb = aLb * L[0], dRb = aRb * R[0];
  SLb += dLb; uLb -= dLb;
  SRb += dRb; uRb -= dRb;
  // SR = max(uL + cL, uR + cR), SL = min(uL - cL, uR - cR)
  T cLb = T(0), cRb = T(0);
  if (pickRa) { uLb += SRb; cLb += SRb; } else { uRb += SRb; cRb += SRb; }
  if (pickLa) { uLb += SLb; cLb -= SLb; } else { uRb += SLb; cRb -= SLb; }
  // cK = sqrt(gamma PK rK)
  const T tLb = cLb * T(0.5) * rcp_(cL), tRb = cRb * T(0.5) * rcp_(cR);
  PLb += tLb * c.gamma * rL;
  PRb += tRb * c.gamma * rR;
  rLb += tLb * c.gamma * L[4];
  rRb += tRb * c.gamma * R[4];
  // rK = 1 / rhoK
  rhoLb -= rLb * rL * rL;
  rhoRb -= rRb * rR * rR;
  Lb[0] += rhoLb; Lb[n] += uLb; Lb[4] += PLb;
  Rb[0] += rhoRb; Rb[n] += uRb; Rb[4] += PRb;
}

// ------------------------------------------------------------------------------------------------
// Two-wave HLL and Rusanov / local Lax-Friedrichs fluxes (PAPER.md:835 lists them beside HLLC; same wave-speed
// estimates, Eq. A3).  Both are F = wL F_L + wR F_R + wU (U_R - U_L):
//   HLL      b- = min(S_L, 0), b+ = max(S_R, 0):  wL = b+/(b+ - b-), wR = -b-/(b+ - b-), wU = b+ b-/(b+ - b-)
//            (b- = 0 gives F_L, b+ = 0 gives F_R: the supersonic branches without a select);
//   Rusanov  a = max(|S_L|, |S_R|):               wL = wR = 1/2, wU = -a/2.
// RS: 1 HLL, 2 Rusanov.
// ------------------------------------------------------------------------------------------------
template <class T, int AX>
__device__ __forceinline__ void phys_flux(const T W[5], const Consts<T>& c, T U[5], T F[5]) {
  constexpr int n = 1 + AX;
  const T rho = W[0], u = W[n];
  const T q = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  const T E = W[4] * c.inv_gm1 + T(0.5) * rho * q;
  const T fm = rho * u;
  U[0] = rho; U[1] = rho * W[1]; U[2] = rho * W[2]; U[3] = rho * W[3]; U[4] = E;
  F[0] = fm; F[1] = fm * W[1]; F[2] = fm * W[2]; F[3] = fm * W[3]; F[4] = u * (E + W[4]);
  F[n] += W[4];
}

// Wb += (dU/dW)^T Ub + (dF/dW)^T Fb
template <class T, int AX>
__device__ __forceinline__ void phys_flux_vjp(const T W[5], const Consts<T>& c, const T Ub[5], const T Fb[5], T Wb[5]) {
  constexpr int n = 1 + AX;
  const T rho = W[0], u = W[n];
  const T q = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  const T E = W[4] * c.inv_gm1 + T(0.5) * rho * q;
  const T fm = rho * u;
  const T Eb = Ub[4] + Fb[4] * u;
  const T fmb = Fb[0] + Fb[1] * W[1] + Fb[2] * W[2] + Fb[3] * W[3];
  const T er = Eb * rho;
  Wb[4] += Fb[4] * u + Fb[n] + Eb * c.inv_gm1;
  Wb[0] += Ub[0] + Ub[1] * W[1] + Ub[2] * W[2] + Ub[3] * W[3] + fmb * u + T(0.5) * Eb * q;
  Wb[1] += Fb[1] * fm + Ub[1] * rho + er * W[1];
  Wb[2] += Fb[2] * fm + Ub[2] * rho + er * W[2];
  Wb[3] += Fb[3] * fm + Ub[3] * rho + er * W[3];
  Wb[n] += Fb[4] * (E + W[4]) + fmb * rho;
}

template <class T, int AX, int RS>
__device__ __forceinline__ void hll_flux(const T L[5], const T R[5], const Consts<T>& c, T F[5]) {
  constexpr int n = 1 + AX;
  const T cL = sqrt_(c.gamma * L[4] * rcp_(L[0])), cR = sqrt_(c.gamma * R[4] * rcp_(R[0]));
  const T SL = min_(L[n] - cL, R[n] - cR);          // Eq. A3
  const T SR = max_(L[n] + cL, R[n] + cR);
  T UL[5], UR[5], FL[5], FR[5];
  phys_flux<T, AX>(L, c, UL, FL);
  phys_flux<T, AX>(R, c, UR, FR);
  T wL, wR, wU;
  if (RS == 1) {
    const T bm = min_(SL, T(0)), bp = max_(SR, T(0));
    const T inv = rcp_(bp - bm);
    wL = bp * inv; wR = -bm * inv; wU = bp * bm * inv;
  } else {
    wL = wR = T(0.5);
    wU = T(-0.5) * max_(abs_(SL), abs_(SR));
  }
#pragma unroll
  for (int f = 0; f < 5; ++f) F[f] = wL * FL[f] + wR * FR[f] + wU * (UR[f] - UL[f]);
}

// (Lb, Rb) += (dF/dL, dF/dR)^T Fb on the branches taken (ties as in the flux: S_L >= 0 -> b- inactive, S_R <= 0 -> b+
// inactive, min / max ties -> first argument, |S_L| >= |S_R| -> S_L carries the Rusanov speed)
template <class T, int AX, int RS>
__device__ __forceinline__ void hll_flux_vjp(const T L[5], const T R[5], const Consts<T>& c, const T Fb[5], T Lb[5], T Rb[5]) {
  constexpr int n = 1 + AX;
  const T cL = sqrt_(c.gamma * L[4] * rcp_(L[0])), cR = sqrt_(c.gamma * R[4] * rcp_(R[0]));
  const T sLa = L[n] - cL, sLb = R[n] - cR, sRa = L[n] + cL, sRb = R[n] + cR;
  const bool pickLa = (sLa <= sLb), pickRa = (sRa >= sRb);
  const T SL = pickLa ? sLa : sLb, SR = pickRa ? sRa : sRb;
  T UL[5], UR[5], FL[5], FR[5];
  phys_flux<T, AX>(L, c, UL, FL);
  phys_flux<T, AX>(R, c, UR, FR);
  T wLb = T(0), wRb = T(0), wUb = T(0);
#pragma unroll
  for (int f = 0; f < 5; ++f) { wLb += Fb[f] * FL[f]; wRb += Fb[f] * FR[f]; wUb += Fb[f] * (UR[f] - UL[f]); }
  T wL, wR, wU, SLb = T(0), SRb = T(0);
  if (RS == 1) {
    const bool onm = (SL < T(0)), onp = (SR > T(0));
    const T bm = onm ? SL : T(0), bp = onp ? SR : T(0);
    const T inv = rcp_(bp - bm);
    wL = bp * inv; wR = -bm * inv; wU = bp * bm * inv;
    const T invb = wLb * bp - wRb * bm + wUb * bp * bm;
    const T db = -invb * inv * inv;
    const T bpb = (wLb + wUb * bm) * inv + db;
    const T bmb = (wUb * bp - wRb) * inv - db;
    if (onp) SRb = bpb;
    if (onm) SLb = bmb;
  } else {
    wL = wR = T(0.5);
    const T aL = abs_(SL), aR = abs_(SR);
    const T a = (aL >= aR) ? aL : aR;
    wU = T(-0.5) * a;
    const T ab = T(-0.5) * wUb;
    if (aL >= aR) SLb = (SL >= T(0)) ? ab : -ab; else SRb = (SR >= T(0)) ? ab : -ab;
  }
  T ULb[5], URb[5], FLb[5], FRb[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) { FLb[f] = wL * Fb[f]; FRb[f] = wR * Fb[f]; URb[f] = wU * Fb[f]; ULb[f] = -URb[f]; }
  phys_flux_vjp<T, AX>(L, c, ULb, FLb, Lb);
  phys_flux_vjp<T, AX>(R, c, URb, FRb, Rb);
  // S_R = max(uL + cL, uR + cR), S_L = min(uL - cL, uR - cR); c_K = sqrt(gamma P_K / rho_K)
  T cLb = T(0), cRb = T(0);
  if (pickRa) { Lb[n] += SRb; cLb += SRb; } else { Rb[n] += SRb; cRb += SRb; }
  if (pickLa) { Lb[n] += SLb; cLb -= SLb; } else { Rb[n] += SLb; cRb -= SLb; }
  const T hL = T(0.5) * cLb * cL, hR = T(0.5) * cRb * cR;
  Lb[4] += hL * rcp_(L[4]); Lb[0] -= hL * rcp_(L[0]);
  Rb[4] += hR * rcp_(R[4]); Rb[0] -= hR * rcp_(R[0]);
}

// RS: 0 HLLC, 1 HLL, 2 Rusanov (DH_OPT_RIEMANN)
template <class T, int AX, int RS>
__device__ __forceinline__ void riemann_flux(const T L[5], const T R[5], const Consts<T>& c, T F[5]) {
  if (RS == 0) hllc<T, AX>(L, R, c, F); else hll_flux<T, AX, (RS == 0 ? 1 : RS)>(L, R, c, F);
}
template <class T, int AX, int RS>
__device__ __forceinline__ void riemann_flux_vjp(const T L[5], const T R[5], const Consts<T>& c, const T Fb[5], T Lb[5], T Rb[5]) {
  if (RS == 0) hllc_vjp<T, AX>(L, R, c, Fb, Lb, Rb); else hll_flux_vjp<T, AX, (RS == 0 ? 1 : RS)>(L, R, c, Fb, Lb, Rb);
}

// ------------------------------------------------------------------------------------------------
// cooling, Eq. 23 with N_sub = 1 and the floor of Eq. 24; only E changes.
// ------------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ T cool_energy(const T U[5], T dt, const Consts<T>& c) {
  const T rho = U[0];
  const T r = rcp_(rho);
  const T Ek = T(0.5) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) * r;
  const T Eth = U[4] - Ek;
  const T Tg = max_(c.gm1 * Eth * r, T(0));
  const T Ta = c.alpha_is_half ? sqrt_(Tg) : ((Tg > T(0)) ? pow_(Tg, c.alpha) : T(0));
  const T Eth1 = max_(rho * c.t_floor * c.inv_gm1, Eth - rho * rho * c.lambda0 * Ta * dt);
  return Ek + Eth1;
}

// gbar = J_cool(U1)^T g  (U1: pre-cooling state).  Only the E row of J differs from the identity.
template <class T>
__device__ __forceinline__ void cool_vjp(const T U[5], T dt, const Consts<T>& c, const T g[5], T gb[5]) {
  const T rho = U[0];
  const T r = rcp_(rho);
  const T m2 = U[1] * U[1] + U[2] * U[2] + U[3] * U[3];
  const T Ek = T(0.5) * m2 * r;
  const T Eth = U[4] - Ek;
  const T Traw = c.gm1 * Eth * r;
  const bool Tpos = (Traw >= T(0));
  const T Tg = Tpos ? Traw : T(0);
  const T Ta = c.alpha_is_half ? sqrt_(Tg) : ((Tg > T(0)) ? pow_(Tg, c.alpha) : T(0));
  const T k = rho * rho * c.lambda0 * dt;
  const T cand = Eth - k * Ta;
  const T Efl = rho * c.t_floor * c.inv_gm1;
  const bool floored = !(Efl < cand);   // max(Efl, cand): ties -> first argument (the floor)
  // Eout = Ek + (floored ? Efl : cand)
  const T gE = g[4];
  T Ekb = gE, rhob = T(0), Ethb = T(0);
  if (floored) {
    rhob += gE * c.t_floor * c.inv_gm1;
  } else {
    Ethb += gE;
    const T dTa = (Tpos && Tg > T(0)) ? c.alpha * Ta * rcp_(Tg) : T(0);   // d T^alpha / dT
    const T Tb = -gE * k * dTa;
    rhob += -gE * T(2) * rho * c.lambda0 * dt * Ta;
    Ethb += Tb * c.gm1 * r;
    rhob += -Tb * Traw * r;
  }
  // Eth = E - Ek;  Ek = m2 / (2 rho)
  Ekb -= Ethb;
  gb[4] = Ethb;
  gb[1] = g[1] + Ekb * U[1] * r;
  gb[2] = g[2] + Ekb * U[2] * r;
  gb[3] = g[3] + Ekb * U[3] * r;
  gb[0] = g[0] + rhob - Ekb * Ek * r;
}

// ------------------------------------------------------------------------------------------------
// The other cooling integrators of PAPER.md:318-325 (reading A20), used by the streaming kernels
// cool_fwd_kernel / cool_vjp_kernel:  cool_mode 0, N_sub > 1: Eq. 23 sub-cycled (rate re-evaluated and the floor of
// Eq. 24 applied every substep);  cool_mode 1: the trapezoid of Eq. 22 with T^pred from the Euler-predicted, floored
// energy.  Edot(E_th) = -rho^2 lambda0 max(T, 0)^alpha,  T = (gamma-1) E_th / rho.
// ------------------------------------------------------------------------------------------------
constexpr int DH_COOL_NSUB_MAX = 64;

// Lambda_CIE(T) of Eq. 19 and d Lambda / dT: interpolation between the nodes, end values held (reading A25)
template <class T>
__device__ __forceinline__ T lambda_table(T Tg, const Consts<T>& c, T& dlam, int& kout, T& wout) {
  const T u = (log2_(Tg) - c.tab_l2t0) * c.tab_inv_dl2t;
  int k = (int)floor_(u);
  k = k < 0 ? 0 : (k > c.ntab - 2 ? c.ntab - 2 : k);
  T w = u - T(k);
  const bool held = (w < T(0)) || (w > T(1));
  w = w < T(0) ? T(0) : (w > T(1) ? T(1) : w);
  const T a = c.tab[k], slope = c.tab[k + 1] - a;
  const T lam = exp2_(a + w * slope);
  dlam = held ? T(0) : lam * slope * c.tab_inv_dl2t * rcp_(Tg);    // d/dT exp2(a + slope (log2 T - l0) / dl)
  kout = k; wout = w;
  return lam;
}

// Edot = n_H Gamma - n_H^2 Lambda (Eqs. 15, 20), n_H = rho, T = (gamma-1) E_th / rho
template <class T>
__device__ __forceinline__ T cool_rate(T Eth, T rho, T r, const Consts<T>& c) {
  const T Traw = c.gm1 * Eth * r;
  const T Tg = max_(Traw, T(0));
  if (c.cool_law == 0) {
    const T Ta = c.alpha_is_half ? sqrt_(Tg) : ((Tg > T(0)) ? pow_(Tg, c.alpha) : T(0));
    return -(rho * rho * c.lambda0) * Ta;
  }
  if (Traw < c.t_switch) {                                  // Eq. 17, lower branch: Eq. 18 and Gamma_0
    const T lam = (Tg > T(0)) ? c.lambda1 * pow_(Tg, c.alpha1) + c.lambda2 * pow_(Tg, c.alpha2) : T(0);
    return rho * c.gamma0 - rho * rho * lam;
  }
  T dlam, w;
  int k;
  return -(rho * rho) * lambda_table(Tg, c, dlam, k, w);
}

// (Ethb, rhob) += (dEdot/dE_th, dEdot/drho) * rateb;  tabacc != NULL: also tabacc[k] += d Edot / d tab[k] * rateb
// (shared-memory accumulator of the table gradient, in the table's own units of log2 Lambda)
template <class T>
__device__ __forceinline__ void cool_rate_vjp(T Eth, T rho, T r, const Consts<T>& c, T rateb, T& Ethb, T& rhob, double* tabacc = nullptr) {
  const T Traw = c.gm1 * Eth * r;
  const bool Tpos = (Traw >= T(0));
  const T Tg = Tpos ? Traw : T(0);
  T lam, dlam, g0 = T(0);                                  // rate = rho g0 - rho^2 lam
  if (c.cool_law == 0) {
    lam = c.lambda0 * (c.alpha_is_half ? sqrt_(Tg) : ((Tg > T(0)) ? pow_(Tg, c.alpha) : T(0)));
    dlam = (Tpos && Tg > T(0)) ? c.alpha * lam * rcp_(Tg) : T(0);
  } else if (Traw < c.t_switch) {
    const T l1 = (Tg > T(0)) ? c.lambda1 * pow_(Tg, c.alpha1) : T(0), l2 = (Tg > T(0)) ? c.lambda2 * pow_(Tg, c.alpha2) : T(0);
    lam = l1 + l2;
    dlam = (Tpos && Tg > T(0)) ? (c.alpha1 * l1 + c.alpha2 * l2) * rcp_(Tg) : T(0);
    g0 = c.gamma0;
  } else {
    int k;
    T w;
    lam = lambda_table(Tg, c, dlam, k, w);
    if (tabacc) {                                          // d lam / d tab[k] = lam ln2 (1 - w), d lam / d tab[k+1] = lam ln2 w
      const double t = -(double)rateb * (double)(rho * rho) * (double)lam * 0.6931471805599453;
      atomicAdd(tabacc + k, t * (1.0 - (double)w));
      atomicAdd(tabacc + k + 1, t * (double)w);
    }
  }
  const T Tb = -rateb * rho * rho * dlam;
  rhob += rateb * (g0 - T(2) * rho * lam);
  Ethb += Tb * c.gm1 * r;
  rhob += -Tb * Traw * r;
}

template <class T>
__device__ __forceinline__ T cool_energy_general(const T U[5], T dt, const Consts<T>& c) {
  const T rho = U[0];
  const T r = rcp_(rho);
  const T Ek = T(0.5) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) * r;
  T Eth = U[4] - Ek;
  const T Efl = rho * c.t_floor * c.inv_gm1;
  int mode = c.cool_mode;
  if (mode == 2) mode = (dt * abs_(cool_rate(Eth, rho, r, c)) > c.f_sub * abs_(Eth)) ? 0 : 1;   // masked choice per cell
  if (mode == 1) {
    const T rn = cool_rate(Eth, rho, r, c);
    const T Ep = max_(Efl, Eth + rn * dt);
    const T rp = cool_rate(Ep, rho, r, c);
    Eth = max_(Efl, Eth + (T(0.5) * dt) * (rn + rp));
  } else {
    const int nsub = c.cool_nsub;
    const T ddt = dt / T(nsub);
    for (int k = 0; k < nsub; ++k) Eth = max_(Efl, Eth + cool_rate(Eth, rho, r, c) * ddt);
  }
  return Ek + Eth;
}

// gbar = J_cool(U1)^T g for the integrators above (U1: pre-cooling state); max(E_floor, x) ties -> the floor
template <class T>
__device__ __forceinline__ void cool_vjp_general(const T U[5], T dt, const Consts<T>& c, const T g[5], T gb[5], double* tabacc = nullptr) {
  const T rho = U[0];
  const T r = rcp_(rho);
  const T Ek = T(0.5) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) * r;
  const T Eth0 = U[4] - Ek;
  const T Efl = rho * c.t_floor * c.inv_gm1;
  const T dfl = c.t_floor * c.inv_gm1;          // dE_floor / drho
  const T gE = g[4];
  T Ethb = T(0), rhob = T(0);                   // cotangents of E_th^0 and rho
  int mode = c.cool_mode;
  if (mode == 2) mode = (dt * abs_(cool_rate(Eth0, rho, r, c)) > c.f_sub * abs_(Eth0)) ? 0 : 1;   // the choice itself has no derivative
  if (mode == 1) {
    const T rn = cool_rate(Eth0, rho, r, c);
    const T candp = Eth0 + rn * dt;
    const bool flp = !(Efl < candp);
    const T Ep = flp ? Efl : candp;
    const T rp = cool_rate(Ep, rho, r, c);
    const T cand = Eth0 + (T(0.5) * dt) * (rn + rp);
    if (!(Efl < cand)) {
      rhob += gE * dfl;
    } else {
      Ethb += gE;
      T rnb = T(0.5) * dt * gE;
      const T rpb = rnb;
      T Epb = T(0);
      cool_rate_vjp(Ep, rho, r, c, rpb, Epb, rhob, tabacc);
      if (flp) rhob += Epb * dfl; else { Ethb += Epb; rnb += Epb * dt; }
      cool_rate_vjp(Eth0, rho, r, c, rnb, Ethb, rhob, tabacc);
    }
  } else {
    const int nsub = c.cool_nsub;
    const T ddt = dt / T(nsub);
    T Es[DH_COOL_NSUB_MAX];                     // E_th^k, k = 0 .. nsub-1
    bool fl_last = false;
    T Eth = Eth0;
    for (int k = 0; k < nsub; ++k) {
      Es[k] = Eth;
      const T cand = Eth + cool_rate(Eth, rho, r, c) * ddt;
      fl_last = !(Efl < cand);
      Eth = fl_last ? Efl : cand;
    }
    T eb = gE;                                  // cotangent of E_th^{k+1}
    for (int k = nsub - 1; k >= 0; --k) {
      const T cand = Es[k] + cool_rate(Es[k], rho, r, c) * ddt;
      if (!(Efl < cand)) { rhob += eb * dfl; eb = T(0); break; }   // floored: nothing earlier matters
      T ekb = eb;
      cool_rate_vjp(Es[k], rho, r, c, eb * ddt, ekb, rhob, tabacc);
      eb = ekb;
    }
    Ethb = eb;
  }
  // E_out = Ek + E_th^N;  E_th^0 = E - Ek;  Ek = |m|^2 / (2 rho)
  const T Ekb = gE - Ethb;
  gb[4] = Ethb;
  gb[1] = g[1] + Ekb * U[1] * r;
  gb[2] = g[2] + Ekb * U[2] * r;
  gb[3] = g[3] + Ekb * U[3] * r;
  gb[0] = g[0] + rhob - Ekb * Ek * r;
}

}  // namespace dh
