// dh_pack.cuh — two-cell "pack" arithmetic for the fused kernels (sm_100a).
//
// The fused stage kernels give every thread TWO cells adjacent in x and run the same instruction stream on
// both.  For fp32 the add / mul / fma of such a pair is ONE packed instruction on sm_100 (PTX add/mul/fma
// .f32x2 -> SASS FADD2 / FMUL2 / FFMA2): the fp32 pipe time is unchanged but the issue slots halve, which
// is what binds this kernel ("Kernels").  min / max / MUFU / select stay per lane.  For fp64
// the pack is two scalars.
#pragma once
#include "dh_math.cuh"

namespace dh {

#define DH_DI __device__ __forceinline__

template <class T> struct P2 { T x, y; };
template <> struct alignas(8) P2<float> { float x, y; };
template <> struct alignas(16) P2<double> { double x, y; };

struct B2 { bool x, y; };

// ---- fp32: packed PTX ----------------------------------------------------------------------------
DH_DI unsigned long long pk_(P2<float> a) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
  return r;
}
DH_DI P2<float> upk_(unsigned long long r) {
  P2<float> a;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
  return a;
}
DH_DI P2<float> add2(P2<float> a, P2<float> b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b)));
  return upk_(r);
}
DH_DI P2<float> sub2(P2<float> a, P2<float> b) {
  unsigned long long r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b)));
  return upk_(r);
}
DH_DI P2<float> mul2(P2<float> a, P2<float> b) {
  unsigned long long r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b)));
  return upk_(r);
}
DH_DI P2<float> fma2(P2<float> a, P2<float> b, P2<float> c) {   // a*b + c
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b)), "l"(pk_(c)));
  return upk_(r);
}
// a*b - c and c - a*b: two scalar FFMA with a free operand negation (no packed negate exists)
DH_DI P2<float> fms2(P2<float> a, P2<float> b, P2<float> c) { return {fmaf(a.x, b.x, -c.x), fmaf(a.y, b.y, -c.y)}; }
DH_DI P2<float> fnma2(P2<float> a, P2<float> b, P2<float> c) { return {fmaf(-a.x, b.x, c.x), fmaf(-a.y, b.y, c.y)}; }
// minmod(a, b) in three ALU-pipe instructions: FMNMX.xorsign.abs gives +-min(|a|,|b|) with the sign positive
// exactly when a and b agree in sign; clamping at 0 kills the disagreeing case; the sign of a is put back.
DH_DI float minmod_(float a, float b) {
  float d;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  d = fmaxf(d, 0.0f);
  return __uint_as_float(__float_as_uint(d) | (__float_as_uint(a) & 0x80000000u));
}
// twice minmod(a, b): the clamp at zero as d + |d| (= 2 d or +0, exact) on the FMA pipe instead of max(d, 0) on the half-rate ALU
// pipe; the face states take the factor back (W +- 0.25 s2 is bit for bit W +- 0.5 s: scaling by a power of two is exact).
// The fused forward kernel is bound by its math-pipe cycles: one ALU instruction (two cycles) becomes one FADD (one).
DH_DI float minmod2x_(float a, float b) {
  float d;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  d = __fadd_rn(d, fabsf(d));
  return __uint_as_float(__float_as_uint(d) | (__float_as_uint(a) & 0x80000000u));
}
DH_DI double minmod_(double a, double b) {
  const double mn = fmin(a, b), mx = fmax(a, b);
  return fmin(fmax(mn, 0.0), mx);
}

// ---- fp64: two scalars ---------------------------------------------------------------------------
// (the _rn intrinsics are never contracted into FMAs, so every call site rounds identically: a face flux has the
// same bits whichever warp computes it, which is what makes the step translation-equivariant bitwise)
DH_DI P2<double> add2(P2<double> a, P2<double> b) { return {__dadd_rn(a.x, b.x), __dadd_rn(a.y, b.y)}; }
DH_DI P2<double> sub2(P2<double> a, P2<double> b) { return {__dsub_rn(a.x, b.x), __dsub_rn(a.y, b.y)}; }
DH_DI P2<double> mul2(P2<double> a, P2<double> b) { return {__dmul_rn(a.x, b.x), __dmul_rn(a.y, b.y)}; }
DH_DI P2<double> fma2(P2<double> a, P2<double> b, P2<double> c) { return {fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)}; }
DH_DI P2<double> fms2(P2<double> a, P2<double> b, P2<double> c) { return {fma(a.x, b.x, -c.x), fma(a.y, b.y, -c.y)}; }
DH_DI P2<double> fnma2(P2<double> a, P2<double> b, P2<double> c) { return {fma(-a.x, b.x, c.x), fma(-a.y, b.y, c.y)}; }

// ---- per-lane operations -------------------------------------------------------------------------
DH_DI float rsqrt_(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
DH_DI double rsqrt_(double x) { return 1.0 / sqrt(x); }

DH_DI float fma_(float a, float b, float c) { return fmaf(a, b, c); }
DH_DI double fma_(double a, double b, double c) { return fma(a, b, c); }
template <class T> DH_DI P2<T> bc2(T s) { return {s, s}; }
template <class T> DH_DI P2<T> min2(P2<T> a, P2<T> b) { return {min_(a.x, b.x), min_(a.y, b.y)}; }
template <class T> DH_DI P2<T> max2(P2<T> a, P2<T> b) { return {max_(a.x, b.x), max_(a.y, b.y)}; }
template <class T> DH_DI P2<T> min2(P2<T> a, T b) { return {min_(a.x, b), min_(a.y, b)}; }
template <class T> DH_DI P2<T> max2(P2<T> a, T b) { return {max_(a.x, b), max_(a.y, b)}; }
template <class T> DH_DI P2<T> rcp2(P2<T> a) { return {rcp_(a.x), rcp_(a.y)}; }
template <class T> DH_DI P2<T> rsqrt2(P2<T> a) { return {rsqrt_(a.x), rsqrt_(a.y)}; }
template <class T> DH_DI P2<T> sel2(B2 m, P2<T> a, P2<T> b) { return {m.x ? a.x : b.x, m.y ? a.y : b.y}; }
template <class T> DH_DI B2 ge2(P2<T> a, T b) { return {a.x >= b, a.y >= b}; }

// ---- scheme pieces on packs ----------------------------------------------------------------------
// primitives of two cells (Eq. 2); same arithmetic as prim() in dh_math.cuh
template <class T>
DH_DI void prim2(const P2<T> U[5], const Consts<T>& c, P2<T> W[5]) {
  const P2<T> rho = max2(U[0], c.rho_floor);
  const P2<T> r = rcp2(rho);
  const P2<T> vx = mul2(U[1], r), vy = mul2(U[2], r), vz = mul2(U[3], r);
  const P2<T> q = fma2(U[3], vz, fma2(U[2], vy, mul2(U[1], vx)));   // |m|^2 / rho
  W[0] = rho; W[1] = vx; W[2] = vy; W[3] = vz;
  W[4] = max2(mul2(bc2(c.gm1), fnma2(bc2(T(0.5)), q, U[4])), c.p_floor);
}

// limited slope of both cells: a = W_{+1} - W, b = W - W_{-1}  (Eq. A1)
template <class T, int LIM>
DH_DI T limit1(T a, T b) {
  if (LIM == 0) return minmod_(a, b);
  return limit<T, LIM>(a, b);
}
template <class T, int LIM>
DH_DI P2<T> limit2(P2<T> a, P2<T> b) { return {limit1<T, LIM>(a.x, b.x), limit1<T, LIM>(a.y, b.y)}; }
// the limited slope scaled by SlopeScale<T, LIM>::k (fp32 minmod: 2, see minmod2x_; everything else: 1); a face state is
// W +- (0.5 / k) s
template <class T, int LIM> struct SlopeScale { static constexpr int k = (LIM == 0 && sizeof(T) == 4) ? 2 : 1; };
template <class T, int LIM>
DH_DI T limit1s(T a, T b) {
  if constexpr (LIM == 0 && sizeof(T) == 4) return minmod2x_(a, b);
  else return limit1<T, LIM>(a, b);
}
template <class T, int LIM>
DH_DI P2<T> limit2s(P2<T> a, P2<T> b) { return {limit1s<T, LIM>(a.x, b.x), limit1s<T, LIM>(a.y, b.y)}; }

// HLLC flux of two faces with normal axis AX (Eq. A3 for the wave speeds); the
// arrangement of hllc() in dh_math.cuh (up to H_K = E_K + P_K being formed in one piece here): star state on the upwind side only, supersonic branches folded
// into S_eff = min(S_L, 0) / max(S_R, 0), transverse momentum flux = v_t * F_mass, one rsqrt per sound
// speed (c = gP * rsqrt(gP * rho)), E_K formed without a density reciprocal.
template <class T, int AX>
DH_DI void hllc2(const P2<T> L[5], const P2<T> R[5], const Consts<T>& c, P2<T> F[5]) {
  constexpr int n = 1 + AX, t1 = 1 + (AX + 1) % 3, t2 = 1 + (AX + 2) % 3;
  const P2<T> g = bc2(c.gamma);
  const P2<T> gPL = mul2(g, L[4]), gPR = mul2(g, R[4]);
  const P2<T> cL = mul2(gPL, rsqrt2(mul2(gPL, L[0]))), cR = mul2(gPR, rsqrt2(mul2(gPR, R[0])));
  const P2<T> uL = L[n], uR = R[n];
  const P2<T> SL = min2(sub2(uL, cL), sub2(uR, cR));          // Eq. A3
  const P2<T> SR = max2(add2(uL, cL), add2(uR, cR));
  const P2<T> dL = sub2(SL, uL), dR = sub2(SR, uR);
  const P2<T> aL = mul2(L[0], dL), aR = mul2(R[0], dR);
  const P2<T> num = fnma2(aR, uR, fma2(aL, uL, sub2(R[4], L[4])));
  const P2<T> Ss = mul2(num, rcp2(sub2(aL, aR)));             // contact speed S*
  const B2 left = ge2(Ss, T(0));
  const P2<T> rhoK = sel2(left, L[0], R[0]), uK = sel2(left, uL, uR);
  const P2<T> v1 = sel2(left, L[t1], R[t1]), v2 = sel2(left, L[t2], R[t2]);
  const P2<T> PK = sel2(left, L[4], R[4]), aK = sel2(left, aL, aR), dK = sel2(left, dL, dR);
  const P2<T> Seff = sel2(left, min2(SL, T(0)), max2(SR, T(0)));   // 0 in the supersonic branches -> F = F_K
  const P2<T> q = fma2(v2, v2, fma2(v1, v1, mul2(uK, uK)));
  // H_K = E_K + P_K in one piece (gamma / (gamma - 1) = 1 + 1 / (gamma - 1)): E_K alone is never needed, and both places that
  // used it added P_K (two packed additions per face pair fewer)
  const P2<T> HK = fma2(mul2(bc2(T(0.5)), rhoK), q, mul2(bc2(c.inv_gm1 + T(1)), PK));
  const P2<T> mK = mul2(rhoK, uK);
  const P2<T> Y = sub2(Ss, uK);
  // star-state jumps in terms of w = (S* - u_K) / (S_K - S*):  rho* - rho = rho w,  (rho u)* - rho u = rho (Y + w S*),
  // E* - E = w (E + P + a_K S*)   (the same algebra as U*_K - U_K of the textbook form, two packed and two scalar
  // instructions shorter per face pair and without the cancellation in E* - E)
  const P2<T> w = mul2(Y, rcp2(sub2(dK, Y)));
  const P2<T> t = mul2(Seff, rhoK);
  const P2<T> Fm = fma2(t, w, mK);
  const P2<T> ZE = fma2(aK, Ss, HK);
  F[0] = Fm;
  F[n] = fma2(t, fma2(w, Ss, Y), fma2(mK, uK, PK));
  F[t1] = mul2(v1, Fm);
  F[t2] = mul2(v2, Fm);
  F[4] = fma2(mul2(Seff, w), ZE, mul2(uK, HK));
}

// HLL (RS = 1) and Rusanov (RS = 2) fluxes of two faces (wave speeds of Eq. A3), the arrangement of
// hll_flux() in dh_math.cuh: F = wL F_L + wR F_R + wU (U_R - U_L) with
//   HLL      b- = min(S_L, 0), b+ = max(S_R, 0):  wL = b+/(b+ - b-), wR = -b-/(b+ - b-), wU = b- wL
//   Rusanov  wL = wR = 1/2, wU = -max(|S_L|, |S_R|)/2.
template <class T, int AX>
DH_DI void phys2(const P2<T> W[5], const Consts<T>& c, P2<T> U[5], P2<T> F[5]) {
  constexpr int n = 1 + AX, t1 = 1 + (AX + 1) % 3, t2 = 1 + (AX + 2) % 3;
  const P2<T> q = fma2(W[3], W[3], fma2(W[2], W[2], mul2(W[1], W[1])));
  const P2<T> E = fma2(mul2(bc2(T(0.5)), W[0]), q, mul2(bc2(c.inv_gm1), W[4]));
  U[0] = W[0]; U[1] = mul2(W[0], W[1]); U[2] = mul2(W[0], W[2]); U[3] = mul2(W[0], W[3]); U[4] = E;
  const P2<T> fm = U[n];
  F[0] = fm;
  F[n] = fma2(fm, W[n], W[4]);
  F[t1] = mul2(fm, W[t1]);
  F[t2] = mul2(fm, W[t2]);
  F[4] = mul2(W[n], add2(E, W[4]));
}

template <class T, int AX, int RS>
DH_DI void hll2(const P2<T> L[5], const P2<T> R[5], const Consts<T>& c, P2<T> F[5]) {
  constexpr int n = 1 + AX;
  const P2<T> g = bc2(c.gamma);
  const P2<T> gPL = mul2(g, L[4]), gPR = mul2(g, R[4]);
  const P2<T> cL = mul2(gPL, rsqrt2(mul2(gPL, L[0]))), cR = mul2(gPR, rsqrt2(mul2(gPR, R[0])));
  const P2<T> SL = min2(sub2(L[n], cL), sub2(R[n], cR));          // Eq. A3
  const P2<T> SR = max2(add2(L[n], cL), add2(R[n], cR));
  P2<T> wL, wR, wU;
  if (RS == 1) {
    const P2<T> bm = min2(SL, T(0)), bp = max2(SR, T(0));
    const P2<T> nbm = {max_(-SL.x, T(0)), max_(-SL.y, T(0))};
    const P2<T> inv = rcp2(add2(bp, nbm));
    wL = mul2(bp, inv); wR = mul2(nbm, inv); wU = mul2(bm, wL);
  } else {
    wL = wR = bc2(T(0.5));
    wU = mul2(bc2(T(-0.5)), P2<T>{max_(abs_(SL.x), abs_(SR.x)), max_(abs_(SL.y), abs_(SR.y))});
  }
  P2<T> UL[5], UR[5], FL[5], FR[5];
  phys2<T, AX>(L, c, UL, FL);
  phys2<T, AX>(R, c, UR, FR);
#pragma unroll
  for (int f = 0; f < 5; ++f) F[f] = fma2(wU, sub2(UR[f], UL[f]), fma2(wL, FL[f], mul2(wR, FR[f])));
}

// RS: 0 HLLC, 1 HLL, 2 Rusanov (DH_OPT_RIEMANN)
template <class T, int AX, int RS>
DH_DI void riemann2(const P2<T> L[5], const P2<T> R[5], const Consts<T>& c, P2<T> F[5]) {
  if (RS == 0) hllc2<T, AX>(L, R, c, F); else hll2<T, AX, (RS == 0 ? 1 : RS)>(L, R, c, F);
}

// cooling of two finished cells (Eqs. 23-24); per lane
// CFL candidate test (dh_advance): an estimate of max_a |v_a| + c_s for the two cells of a pack of CONSERVED values in
// fast math (Eq. A8; dh_cfl.cu evaluates the exact recipe on the packs that pass).  No selects: the pressure floor
// enters as a sum on top of max(e_int, 0) (an upper bound of the recipe's max(P, P_floor)), a density at or below zero
// and any NaN / Inf turn the estimate into NaN or Inf, and `!(s < thr)` makes such a pack a candidate.
template <class T>
DH_DI bool cfl_candidate2(const P2<T> U[5], const Consts<T>& c, T thr) {
  const P2<T> r = rcp2(U[0]);
  const P2<T> q = fma2(U[3], U[3], fma2(U[2], U[2], mul2(U[1], U[1])));
  // an internal energy between -p_floor / (gamma - 1) and 0 must not lower the estimate below the recipe's floored
  // pressure: clamp it at zero before the floor is added (a negative e_int is then simply a floored cell)
  // (a select, not a max: a NaN must stay a NaN; E = -Inf would be clamped away, so 0 * E, which is NaN for any
  // non-finite E, rides on the floor term)
  const P2<T> er = fma2(bc2(T(-0.5)), mul2(q, r), U[4]);
  const P2<T> ei = {er.x < T(0) ? T(0) : er.x, er.y < T(0) ? T(0) : er.y};
  const P2<T> c2 = mul2(fma2(bc2(c.gamma * c.gm1), ei, fma2(U[4], bc2(T(0)), bc2(c.gamma * c.p_floor))), r);
  const P2<T> cs = mul2(c2, rsqrt2(c2));
  const T mx = max_(max_(abs_(U[1].x), abs_(U[2].x)), abs_(U[3].x));
  const T my = max_(max_(abs_(U[1].y), abs_(U[2].y)), abs_(U[3].y));
  const T sx = fma_(mx, r.x, cs.x), sy = fma_(my, r.y, cs.y);
  return !(sx < thr) || !(sy < thr);
}

template <class T>
DH_DI void cool2(P2<T> U[5], T dt, const Consts<T>& c) {
  T a[5] = {U[0].x, U[1].x, U[2].x, U[3].x, U[4].x};
  T b[5] = {U[0].y, U[1].y, U[2].y, U[3].y, U[4].y};
  U[4].x = cool_energy(a, dt, c);
  U[4].y = cool_energy(b, dt, c);
}

}  // namespace dh
