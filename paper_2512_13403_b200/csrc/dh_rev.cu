// dh_rev.cu — fused reverse-mode stage (step a7 of SURVEY.md §8(a), dt constant per PAPER.md:876).
//
// One reversed stage  out = w1 b1 + w2 b2 - tau J_D(U)^T g  (D(U) = sum_a (F_{a,+1/2} - F_{a,-1/2}) / dx_a, Eq. A4) is the
// transpose of: primitives -> minmod slopes -> face states -> HLLC flux -> flux difference.  Written per axis for
// cell i (coef = tau / dx_a):
//     lambda_{i+1/2} = coef (g_{i+1} - g_i)                                   face cotangent
//     (Lb, Rb)_{i+1/2} = J_HLLC(L_i, R_{i+1})^T lambda_{i+1/2}                one HLLC adjoint per face
//     T_i = Lb_{i+1/2} + Rb_{i-1/2},   S_i = (Lb_{i+1/2} - Rb_{i-1/2}) / 2    state and slope cotangents
//     minmod(a_i, b_i) passes S_i to a_i (if |a| <= |b|) or to b_i, or to neither (a b <= 0):
//     Wb_i = T_i + [b-branch: +S_i | a-branch: -S_i]  +  (a-branch S_{i-1})  -  (b-branch S_{i+1})
//     Ub_i = (dW/dU)_i^T Wb_i
// The last two terms of Wb_i come from the neighbours' slopes, i.e. they depend on faces i-3/2 .. i+3/2.  Doing
// everything in one kernel would make every tile recompute two extra layers of face adjoints around itself; the
// one-thread-per-cell gather kernel (dh_naive.cu) does exactly that and spends 12 HLLC adjoints per cell.  Here
// the work is split in two launches that share a scratch slab:
//   A  rev_faces_kernel   fused z-sweep (7 row warps x one pack + helper; z in registers, x / y through shared planes,
//                         R states of the neighbouring cells recomputed locally, ONE block barrier per plane): every
//                         face adjoint once.  The neighbour terms along x are exchanged inside the warp (shuffles of the
//                         masked slope cotangent c = S masked by a b > 0, branch flag in the mantissa LSB, <= 1 ulp) and
//                         those along z stay in the sweep (a cell is stored one plane after its own z terms are known), so
//                         per cell it writes  Wp = everything but the y neighbour terms  and  c^y; the x terms that cross a
//                         tile edge go through a thin array of the tile rows' first and last c^x;
//   B  rev_gather_kernel  streaming: Wb_i = Wp_i + [a-branch c^y_{j-1}] - [b-branch c^y_{j+1}] (+ the tile-edge x term),
//                         then Ub = prim_vjp(U, Wb) + w1 b1 + w2 b2.
// Scratch is 10 words per cell of a z slab (+ 10 / 64 for the tile edges); the API layer walks the slabs.  minmod only
// (the branch flag is one bit); other limiters take the gather kernels.  No atomics; deterministic.
#include "dh_internal.cuh"
#include "dh_pack.cuh"

namespace dh {

namespace {

constexpr int RTX = 64;        // cells per tile row = 32 lanes x 2
constexpr int RSW = RTX + 4;   // row pitch of the shared planes (halo 2 on both sides)
constexpr int RXP = 34;        // pitch of the x exchange arrays (33 used)

template <int NW> struct GeoR {
  static constexpr int TY = NW - 1;
  static constexpr int SR = TY + 4;                       // rows of a shared plane
  static constexpr int PLANE = 5 * SR * RSW;              // one buffered plane (all 5 fields)
  static constexpr int XARR = 5 * TY * RXP;
  static constexpr int YARR = 5 * (TY + 1) * RTX;
  static constexpr int STAGE = 5 * TY * RTX;              // cp.async staging of one raw plane of the tile
  static constexpr int NPARK = 11;                        // staging of the next raw plane + 7 parked carries (+ 3 for the second
                                                          // branch factor of the limiters other than minmod)
  static constexpr int TOTAL = 4 * PLANE + 2 * XARR + 2 * YARR + NPARK * STAGE;
  static constexpr int NHALO = 4 * (RSW / 2) + 2 * TY;    // halo packs per plane
  static constexpr int HP = (NHALO + 31) / 32;            // halo packs per helper lane
};

DH_DI int wrapr(int i, int n) {   // i mod n for any i
  int r = i % n;
  return r < 0 ? r + n : r;
}

template <class T> DH_DI P2<T> rlds2(const T* p) { return *reinterpret_cast<const P2<T>*>(p); }
template <class T> DH_DI void rsts2(T* p, P2<T> v) { *reinterpret_cast<P2<T>*>(p) = v; }
template <class T> DH_DI P2<T> rldg2(const T* p) { return *reinterpret_cast<const P2<T>*>(p); }
template <class T> DH_DI void rstg2(T* p, P2<T> v) { *reinterpret_cast<P2<T>*>(p) = v; }

template <class T> DH_DI void rcp_async_pack(T* smem_dst, const T* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (sizeof(T) == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
DH_DI void rcp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
DH_DI void rcp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// branch flag in the mantissa LSB of the masked slope cotangent (written by enc_sign below)
DH_DI bool dec_flag(float v) { return (__float_as_uint(v) & 1u) != 0u; }
DH_DI bool dec_flag(double v) { return (__double_as_longlong(v) & 1ll) != 0ll; }

// minmod branch of slope (a, b) as a factor: 0 if the slope is inactive (a b <= 0), -1/2 on the a-branch
// (|a| <= |b|), +1/2 on the b-branch (reading A7).  With D = Lb - Rbn (so S = D / 2): the cell's own-branch term is
// k D, the masked slope cotangent is |k| D, and the a-branch flag is the sign bit of k.
template <class T> DH_DI T kfac(T a, T b) {
  const T k = (abs_(a) <= abs_(b)) ? T(-0.5) : T(0.5);
  return (a * b > T(0)) ? k : T(0);
}
template <class T> DH_DI P2<T> kfac2(P2<T> a, P2<T> b) { return {kfac(a.x, b.x), kfac(a.y, b.y)}; }
DH_DI float enc_sign(float v, float k) { return __uint_as_float((__float_as_uint(v) & ~1u) | (__float_as_uint(k) >> 31)); }
DH_DI double enc_sign(double v, double k) {
  return __longlong_as_double((__double_as_longlong(v) & ~1ll) | (long long)((unsigned long long)__double_as_longlong(k) >> 63));
}
// cell cotangents of one axis from the two face adjoints of two cells: wp = T + own-branch term, ce = encoded c
template <class T> DH_DI void cell_terms2(P2<T> Lb, P2<T> Rbn, P2<T> k, P2<T>& wp, P2<T>& ce) {
  const P2<T> D = sub2(Lb, Rbn);
  wp = fma2(k, D, add2(Lb, Rbn));
  const P2<T> c = mul2(P2<T>{abs_(k.x), abs_(k.y)}, D);
  ce = {enc_sign(c.x, k.x), enc_sign(c.y, k.y)};
}

// the same with the neighbour terms as plain values instead of the encoded c (used where they stay inside the kernel):
// P = what the next cell along the axis receives (a-branch: S), M = what the previous cell loses (b-branch: S)
template <class T> DH_DI void cell_terms_pm2(P2<T> Lb, P2<T> Rbn, P2<T> k, P2<T>& wp, P2<T>& P, P2<T>& M) {
  const P2<T> D = sub2(Lb, Rbn);
  wp = fma2(k, D, add2(Lb, Rbn));
  P = mul2(P2<T>{max_(-k.x, T(0)), max_(-k.y, T(0))}, D);
  M = mul2(max2(k, T(0)), D);
}

// HLLC adjoint of two faces: the scalar routine of dh_math.cuh on each half of the packs.  The loop over the halves
// is deliberately NOT unrolled: with six inlined copies the body of the plane loop is ~34 KB of code, and the
// profile (profiles/r01c) showed 30 % of the issue slots lost to instruction fetch; rolled up it is ~20 KB.
template <class T, int AX>
DH_DI void hllc_vjp2(const P2<T> L[5], const P2<T> R[5], const Consts<T>& c, const P2<T> Fb[5], P2<T> Lb[5], P2<T> Rb[5]) {
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    T l[5], r[5], fb[5], lb[5], rb[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      l[f] = h ? L[f].y : L[f].x; r[f] = h ? R[f].y : R[f].x; fb[f] = h ? Fb[f].y : Fb[f].x;
      lb[f] = T(0); rb[f] = T(0);
    }
    hllc_vjp<T, AX>(l, r, c, fb, lb, rb);
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      if (h) { Lb[f].y = lb[f]; Rb[f].y = rb[f]; } else { Lb[f].x = lb[f]; Rb[f].x = rb[f]; }
    }
  }
}

// the same for any Riemann flux (RS: 0 HLLC, 1 HLL, 2 Rusanov): riemann_flux_vjp() of dh_math.cuh on each half
template <class T, int AX, int RS>
DH_DI void riemann_vjp2(const P2<T> L[5], const P2<T> R[5], const Consts<T>& c, const P2<T> Fb[5], P2<T> Lb[5], P2<T> Rb[5]) {
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    T l[5], r[5], fb[5], lb[5], rb[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      l[f] = h ? L[f].y : L[f].x; r[f] = h ? R[f].y : R[f].x; fb[f] = h ? Fb[f].y : Fb[f].x;
      lb[f] = T(0); rb[f] = T(0);
    }
    riemann_flux_vjp<T, AX, RS>(l, r, c, fb, lb, rb);
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      if (h) { Lb[f].y = lb[f]; Rb[f].y = rb[f]; } else { Lb[f].x = lb[f]; Rb[f].x = rb[f]; }
    }
  }
}

template <class T> DH_DI P2<T> neg2(P2<T> a) { return {-a.x, -a.y}; }
template <class T> DH_DI P2<T> zsel2(B2 m, P2<T> a) { return {m.x ? a.x : T(0), m.y ? a.y : T(0)}; }

// HLLC adjoint of two faces at once: hllc_vjp() of dh_math.cuh statement by statement on packs, so that the
// multiplies / adds / FMAs issue as packed fp32 instructions; selects, compares and MUFU stay per lane.
template <class T, int AX>
DH_DI void hllc_vjp2p(const P2<T> L[5], const P2<T> R[5], const Consts<T>& c, const P2<T> Fb[5], P2<T> Lb[5], P2<T> Rb[5]) {
  constexpr int n = 1 + AX, t1 = 1 + (AX + 1) % 3, t2 = 1 + (AX + 2) % 3;
  const P2<T> g = bc2(c.gamma), ig = bc2(c.inv_gm1), hf = bc2(T(0.5));
  // ---- forward recompute
  const P2<T> rL = rcp2(L[0]), rR = rcp2(R[0]);
  const P2<T> cL2 = mul2(mul2(g, L[4]), rL), cR2 = mul2(mul2(g, R[4]), rR);
  const P2<T> cL = {sqrt_(cL2.x), sqrt_(cL2.y)}, cR = {sqrt_(cR2.x), sqrt_(cR2.y)};
  const P2<T> uL = L[n], uR = R[n];
  const P2<T> sLa = sub2(uL, cL), sLb = sub2(uR, cR), sRa = add2(uL, cL), sRb = add2(uR, cR);
  const B2 pickLa = {sLa.x <= sLb.x, sLa.y <= sLb.y}, pickRa = {sRa.x >= sRb.x, sRa.y >= sRb.y};
  const P2<T> SL = sel2(pickLa, sLa, sLb), SR = sel2(pickRa, sRa, sRb);
  const P2<T> dL = sub2(SL, uL), dR = sub2(SR, uR);
  const P2<T> aL = mul2(L[0], dL), aR = mul2(R[0], dR);
  const P2<T> num = fma2(neg2(aR), uR, fma2(aL, uL, sub2(R[4], L[4])));
  const P2<T> iden = rcp2(sub2(aL, aR));
  const P2<T> Ss = mul2(num, iden);
  const B2 left = ge2(Ss, T(0)), right = {!left.x, !left.y};
  const P2<T> rhoK = sel2(left, L[0], R[0]), uK = sel2(left, uL, uR), v1 = sel2(left, L[t1], R[t1]), v2 = sel2(left, L[t2], R[t2]);
  const P2<T> PK = sel2(left, L[4], R[4]), SK = sel2(left, SL, SR), aK = sel2(left, aL, aR), rK = sel2(left, rL, rR);
  const B2 seff_on = {left.x ? (SK.x < T(0)) : (SK.x > T(0)), left.y ? (SK.y < T(0)) : (SK.y > T(0))};
  const P2<T> Seff = zsel2(seff_on, SK);
  const P2<T> e = fma2(mul2(PK, rK), ig, mul2(hf, fma2(v2, v2, fma2(v1, v1, mul2(uK, uK)))));
  const P2<T> EK = mul2(rhoK, e), mK = mul2(rhoK, uK);
  const P2<T> inv = rcp2(sub2(SK, Ss));
  const P2<T> fac = mul2(aK, inv);
  const P2<T> Fm = fma2(Seff, sub2(fac, rhoK), mK);
  const P2<T> Y = sub2(Ss, uK), Z = fma2(aK, Ss, PK);
  const P2<T> X = fma2(Y, Z, mul2(aK, e));
  const P2<T> Es = mul2(inv, X);
  // ---- reverse
  const P2<T> Fmb = fma2(Fb[t2], v2, fma2(Fb[t1], v1, Fb[0]));     // F_t = v_t * F_m
  P2<T> v1b = mul2(Fb[t1], Fm), v2b = mul2(Fb[t2], Fm);
  P2<T> uKb = mul2(Fb[4], add2(EK, PK));                            // F_E = uK (EK + PK) + Seff (Es - EK)
  P2<T> EKb = mul2(Fb[4], sub2(uK, Seff));
  P2<T> PKb = mul2(Fb[4], uK);
  P2<T> Seffb = mul2(Fb[4], sub2(Es, EK));
  const P2<T> Esb = mul2(Fb[4], Seff);
  P2<T> invb = mul2(Esb, X);                                        // Es = inv * X,  X = aK e + Y Z
  const P2<T> Xb = mul2(Esb, inv);
  P2<T> aKb = mul2(Xb, e);
  P2<T> eb = mul2(Xb, aK);
  const P2<T> Yb = mul2(Xb, Z), Zb = mul2(Xb, Y);
  P2<T> Ssb = Yb;
  uKb = sub2(uKb, Yb);
  aKb = fma2(Zb, Ss, aKb);
  Ssb = fma2(Zb, aK, Ssb);
  PKb = add2(PKb, Zb);
  P2<T> mKb = mul2(Fb[n], sub2(uK, Seff));                          // F_n = mK uK + PK + Seff (fac Ss - mK)
  uKb = fma2(Fb[n], mK, uKb);
  PKb = add2(PKb, Fb[n]);
  Seffb = fma2(Fb[n], fma2(fac, Ss, neg2(mK)), Seffb);
  const P2<T> FnS = mul2(Fb[n], Seff);
  P2<T> facb = mul2(FnS, Ss);
  Ssb = fma2(FnS, fac, Ssb);
  mKb = add2(mKb, Fmb);                                             // F_m = mK + Seff (fac - rhoK)
  Seffb = fma2(Fmb, sub2(fac, rhoK), Seffb);
  facb = fma2(Fmb, Seff, facb);
  P2<T> rhoKb = neg2(mul2(Fmb, Seff));
  aKb = fma2(facb, inv, aKb);                                       // fac = aK inv; inv = 1 / (SK - Ss)
  invb = fma2(facb, aK, invb);
  const P2<T> wb = neg2(mul2(mul2(invb, inv), inv));
  P2<T> SKb = wb;
  Ssb = sub2(Ssb, wb);
  rhoKb = fma2(mKb, uK, rhoKb);                                     // mK = rhoK uK; EK = rhoK e; e = PK rK / (gamma-1) + q/2
  uKb = fma2(mKb, rhoK, uKb);
  rhoKb = fma2(EKb, e, rhoKb);
  eb = fma2(EKb, rhoK, eb);
  const P2<T> ebg = mul2(eb, ig);
  PKb = fma2(ebg, rK, PKb);
  const P2<T> rKb = mul2(ebg, PK);
  uKb = fma2(eb, uK, uKb);
  v1b = fma2(eb, v1, v1b);
  v2b = fma2(eb, v2, v2b);
  SKb = add2(SKb, zsel2(seff_on, Seffb));                           // Seff = SK on its active branch
  // un-select K
  P2<T> rhoLb = zsel2(left, rhoKb), rhoRb = zsel2(right, rhoKb), uLb = zsel2(left, uKb), uRb = zsel2(right, uKb);
  P2<T> PLb = zsel2(left, PKb), PRb = zsel2(right, PKb), SLb = zsel2(left, SKb), SRb = zsel2(right, SKb);
  P2<T> aLb = zsel2(left, aKb), aRb = zsel2(right, aKb), rLb = zsel2(left, rKb), rRb = zsel2(right, rKb);
  Lb[t1] = zsel2(left, v1b); Rb[t1] = zsel2(right, v1b);
  Lb[t2] = zsel2(left, v2b); Rb[t2] = zsel2(right, v2b);
  const P2<T> numb = mul2(Ssb, iden);                               // Ss = num / den
  const P2<T> denb = neg2(mul2(mul2(Ssb, Ss), iden));
  aLb = add2(aLb, fma2(numb, uL, denb));
  aRb = sub2(aRb, fma2(numb, uR, denb));
  PRb = add2(PRb, numb);
  PLb = sub2(PLb, numb);
  uLb = fma2(numb, aL, uLb);
  uRb = fma2(neg2(numb), aR, uRb);
  rhoLb = fma2(aLb, dL, rhoLb);                                     // aL = rhoL dL, dL = SL - uL (and R)
  rhoRb = fma2(aRb, dR, rhoRb);
  const P2<T> dLb = mul2(aLb, L[0]), dRb = mul2(aRb, R[0]);
  SLb = add2(SLb, dLb); uLb = sub2(uLb, dLb);
  SRb = add2(SRb, dRb); uRb = sub2(uRb, dRb);
  const B2 npRa = {!pickRa.x, !pickRa.y}, npLa = {!pickLa.x, !pickLa.y};   // SR = max(...), SL = min(...)
  uLb = add2(uLb, add2(zsel2(pickRa, SRb), zsel2(pickLa, SLb)));
  uRb = add2(uRb, add2(zsel2(npRa, SRb), zsel2(npLa, SLb)));
  const P2<T> cLb = sub2(zsel2(pickRa, SRb), zsel2(pickLa, SLb));
  const P2<T> cRb = sub2(zsel2(npRa, SRb), zsel2(npLa, SLb));
  const P2<T> tLb = mul2(mul2(cLb, hf), rcp2(cL)), tRb = mul2(mul2(cRb, hf), rcp2(cR));   // cK = sqrt(gamma PK rK)
  const P2<T> tLg = mul2(tLb, g), tRg = mul2(tRb, g);
  PLb = fma2(tLg, rL, PLb);
  PRb = fma2(tRg, rR, PRb);
  rLb = fma2(tLg, L[4], rLb);
  rRb = fma2(tRg, R[4], rRb);
  rhoLb = fma2(neg2(rLb), mul2(rL, rL), rhoLb);                     // rK = 1 / rhoK
  rhoRb = fma2(neg2(rRb), mul2(rR, rR), rhoRb);
  Lb[0] = rhoLb; Lb[n] = uLb; Lb[4] = PLb;
  Rb[0] = rhoRb; Rb[n] = uRb; Rb[4] = PRb;
}

}  // namespace

// The two halved partial derivatives of the limiter on the branch taken, ha = (d lim / da) / 2, hb = (d lim / db) / 2
// (a = W_{i+1} - W_i, b = W_i - W_{i-1}): with D = Lb - Rbn (S = D / 2) cell i keeps (hb - ha) D, cell i+1 receives ha D and
// cell i-1 loses hb D.  minmod has (ha, hb) in {(0,0), (1/2,0), (0,1/2)} and travels as the single factor k = hb - ha
// (kfac above); van Leer and MC carry both.
template <class T, int LIM> DH_DI void hfac(T a, T b, T& ha, T& hb) {
  T da, db;
  limit_grad<T, LIM>(a, b, da, db);
  ha = T(0.5) * da; hb = T(0.5) * db;
}
// park / fetch the factors of the two cells of a pack (LIM == 0: one array, k; else two arrays)
template <class T, int LIM> DH_DI void park_h(T* pk, T* pkb, P2<T> a, P2<T> b) {
  if (LIM == 0) { rsts2(pk, kfac2(a, b)); return; }
  P2<T> ha, hb;
  hfac<T, LIM>(a.x, b.x, ha.x, hb.x);
  hfac<T, LIM>(a.y, b.y, ha.y, hb.y);
  rsts2(pk, ha); rsts2(pkb, hb);
}
template <class T, int LIM> DH_DI void fetch_h(const T* pk, const T* pkb, P2<T>& ha, P2<T>& hb) {
  if (LIM == 0) {
    const P2<T> k = rlds2(pk);
    ha = {max_(-k.x, T(0)), max_(-k.y, T(0))};
    hb = max2(k, T(0));
  } else {
    ha = rlds2(pk); hb = rlds2(pkb);
  }
}
// cell cotangents of one axis: wp = T + own-branch term, P = what the next cell receives, M = what the previous cell loses
template <class T> DH_DI void cell_terms_h2(P2<T> Lb, P2<T> Rbn, P2<T> ha, P2<T> hb, P2<T>& wp, P2<T>& P, P2<T>& M) {
  const P2<T> D = sub2(Lb, Rbn);
  wp = fma2(sub2(hb, ha), D, add2(Lb, Rbn));
  P = mul2(ha, D);
  M = mul2(hb, D);
}

// neighbour terms of an encoded masked slope cotangent c (flag in the LSB = a-branch): what cell i+1 receives from
// cell i (+c on the a-branch) and what cell i-1 receives from cell i (-c on the b-branch; an inactive slope has c = 0)
template <class T> DH_DI T pterm(T c) { return dec_flag(c) ? c : T(0); }
template <class T> DH_DI T mterm(T c) { return dec_flag(c) ? T(0) : c; }
template <class T> DH_DI P2<T> pterm2(P2<T> c) { return {pterm(c.x), pterm(c.y)}; }
template <class T> DH_DI P2<T> mterm2(P2<T> c) { return {mterm(c.x), mterm(c.y)}; }
DH_DI float shfl_up1(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
DH_DI float shfl_dn1(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }
DH_DI double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
DH_DI double shfl_dn1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// ------------------------------------------------------------------------------------------------ kernel A
// Planes in flight at iteration `it` (plane p = first - 3 + it is loaded; `first` = first output plane of the block):
//   p      raw state -> primitives -> shared plane; cotangent -> shared plane
//   p-1    x and y face adjoints; after the block barrier its x terms are completed inside the warp (shuffles; the
//          helper supplies the two cells beside the tile), its own y terms are added, its c^y goes to the scratch
//   p-2    the z face above it is adjoined: its own z terms and the a-branch term of plane p-3 join the parked sum
//   p-3    receives the b-branch term of plane p-2 and is stored: Wp' = everything except the y neighbour terms
template <class T, int NW, int LIM, int RS>
__global__ void __launch_bounds__(NW * 32, 1)
rev_faces_kernel(const RevFaceParams<T> p, const int ZL) {
  using G = GeoR<NW>;
  constexpr int TY = G::TY, SR = G::SR, FP = SR * RSW, FS = TY * RTX;
  constexpr int XF = TY * RXP, YF = (TY + 1) * RTX;       // field pitches of the exchange arrays
  extern __shared__ __align__(16) unsigned char smem_rev[];
  T* const Wsm = reinterpret_cast<T*>(smem_rev);   // [2][5][SR][RSW]  primitive planes p (it&1) and p-1
  T* const Gsm = Wsm + 2 * G::PLANE;               // [2][5][SR][RSW]  cotangent planes p and p-1
  T* const Rxs = Gsm + 2 * G::PLANE;               // [2][5][TY][RXP]   Rb of the face LEFT of lane l's pack (slot 0: helper), by iteration parity
  T* const Rys = Rxs + 2 * G::XARR;                // [2][5][TY+1][RTX] Rb of the face BELOW row r (slot 0: helper), by iteration parity
  T* const Ust = Rys + 2 * G::YARR;                // [NPARK][5][TY][RTX] raw U of the next plane (cp.async) and parked carries (private slots)

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const size_t NP = (size_t)nx * ny, N = NP * nz, SPN = (size_t)p.SP * NP;
  const int x0 = blockIdx.x * RTX, y0 = blockIdx.y * TY;
  const int zrel0 = blockIdx.z * ZL;               // first output plane of this block, relative to p.zs
  const int zl = min(ZL, p.nout - zrel0);
  const int nit = zl + 6;                          // planes first-3 .. first+zl+2
  const P2<T> cx = bc2(p.coef[0]), cy = bc2(p.coef[1]), cz = bc2(p.coef[2]);
  const P2<T> half = bc2(T(0.5)), nhalf = bc2(T(-0.5));
  const Consts<T>& c = p.c;
  int pz = wrapr(p.zs + zrel0 - 3, nz);

  if (w < TY) {
    // ------------------------------------------------------------------------------------ row warp
    const int r = w;
    const size_t o = (size_t)wrapr(y0 + r, ny) * nx + wrapr(x0 + 2 * lane, nx);
    const bool store_ok = (x0 + 2 * lane < nx) && (y0 + r < ny);
    const int so = (r + 2) * RSW + 2 * lane + 2;   // own pack inside a shared plane
    const int xo = r * RXP + lane, yo = r * RTX + 2 * lane;
    T* const ust = Ust + yo;
    T* const pk1 = Ust + G::STAGE + yo;            // parked carries (private slots): Rb of the lower z face
    T* const pk2 = Ust + 2 * G::STAGE + yo;        //   x (complete) + own y terms of plane p-1
    T* const pkx = Ust + 3 * G::STAGE + yo;        //   minmod branch factors of the own cells: x, y, z
    T* const pky = Ust + 4 * G::STAGE + yo;
    T* const pkz = Ust + 5 * G::STAGE + yo;
    T* const pkw = Ust + 6 * G::STAGE + yo;        //   sum of plane p-2 (still missing the b-branch term of the plane above)
    T* const pkc = Ust + 7 * G::STAGE + yo;        //   a-branch z term of plane p-2 (for plane p-1)
    T* const pkxb = Ust + 8 * G::STAGE + yo;       //   second branch factors (limiters other than minmod)
    T* const pkyb = Ust + 9 * G::STAGE + yo;
    T* const pkzb = Ust + 10 * G::STAGE + yo;
    P2<T> Wprev[5], dprev[5], Lz[5], gpp[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      Wprev[f] = dprev[f] = Lz[f] = gpp[f] = bc2(T(0));
      rsts2(pk1 + f * FS, bc2(T(0))); rsts2(pk2 + f * FS, bc2(T(0))); rsts2(pkz + f * FS, bc2(T(0))); rsts2(pkzb + f * FS, bc2(T(0)));
      rsts2(pkw + f * FS, bc2(T(0))); rsts2(pkc + f * FS, bc2(T(0)));
    }
    size_t op = (size_t)pz * NP + o;
#pragma unroll
    for (int f = 0; f < 5; ++f) rcp_async_pack(ust + f * FS, p.U + f * N + op);
    rcp_async_commit();
    rcp_async_wait_all();
    // scratch offset of the plane stored in iteration `it` (plane p-3): advanced by NP per iteration
    long long os3 = ((long long)p.sp0 + zrel0 - 6) * (long long)NP + (long long)o;

#pragma unroll 1
    for (int it = 0; it < nit; ++it) {
      const int bp = it & 1, bq = bp ^ 1;
      T* const Wp_s = Wsm + bp * G::PLANE;
      const T* const Wq_s = Wsm + bq * G::PLANE;
      const T* const Gq_s = Gsm + bq * G::PLANE;
      const bool xy = (it >= 4) && (it <= zl + 3);   // plane p-1 is an output plane: its c^y is wanted
      P2<T> Uc[5];
#pragma unroll
      for (int f = 0; f < 5; ++f) Uc[f] = rlds2(ust + f * FS);
      // cotangent of plane p straight into its shared plane (read by the neighbours in the next iteration), and the
      // raw state of plane p+1 into the staging slots; both are waited for at the end of the iteration
      int pzn = pz + 1;
      size_t opn = op + NP;
      if (pzn == nz) { pzn = 0; opn = o; }
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        rcp_async_pack(Gsm + bp * G::PLANE + f * FP + so, p.g + f * N + op);
        rcp_async_pack(ust + f * FS, p.U + f * N + opn);
      }
      rcp_async_commit();
      P2<T> Wn[5];
      prim2(Uc, c, Wn);
#pragma unroll
      for (int f = 0; f < 5; ++f) rsts2(Wp_s + f * FP + so, Wn[f]);
      P2<T> gq[5];                                  // own cotangent of plane p-1
#pragma unroll
      for (int f = 0; f < 5; ++f) gq[f] = rlds2(Gq_s + f * FP + so);

      // ---- z: slope of plane p-1, adjoint of the face between p-2 and p-1, which completes the z terms of plane p-2
      {
        P2<T> Rz[5], lam[5], Lb[5], Rb[5];
        P2<T> az[5], bz[5];                          // the differences of plane p-1's slopes, for its branch factors
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const P2<T> a = sub2(Wn[f], Wprev[f]);
          const P2<T> s = limit2<T, LIM>(a, dprev[f]);
          az[f] = a; bz[f] = dprev[f];
          Rz[f] = fma2(nhalf, s, Wprev[f]);
          Wn[f] = fma2(half, s, Wprev[f]);           // left state of the NEXT z face
          dprev[f] = a;
          lam[f] = mul2(cz, sub2(gq[f], gpp[f]));
          gpp[f] = gq[f];
        }
        if (RS == 0) hllc_vjp2p<T, 2>(Lz, Rz, c, lam, Lb, Rb); else riemann_vjp2<T, 2, RS>(Lz, Rz, c, lam, Lb, Rb);
        const bool stz = (it >= 6) && store_ok;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          Lz[f] = Wn[f];
          P2<T> wp, Pz, Mz;
          if (LIM == 0) {
            cell_terms_pm2(Lb[f], rlds2(pk1 + f * FS), rlds2(pkz + f * FS), wp, Pz, Mz);   // cell of plane p-2: parked Rb and factor
          } else {
            P2<T> ha, hb;
            fetch_h<T, LIM>(pkz + f * FS, pkzb + f * FS, ha, hb);
            cell_terms_h2(Lb[f], rlds2(pk1 + f * FS), ha, hb, wp, Pz, Mz);
          }
          rsts2(pk1 + f * FS, Rb[f]);
          park_h<T, LIM>(pkz + f * FS, pkzb + f * FS, az[f], bz[f]);
          const P2<T> Pprev = rlds2(pkc + f * FS);                                // a-branch term of plane p-3 for plane p-2
          const P2<T> fin = sub2(rlds2(pkw + f * FS), Mz);                        // plane p-3 is complete (but for y)
          rsts2(pkw + f * FS, add2(add2(wp, rlds2(pk2 + f * FS)), Pprev));
          rsts2(pkc + f * FS, Pz);
          if (stz) rstg2(p.Wp + f * SPN + os3, fin);
        }
      }

      // ---- x / y on plane p-1: slopes of the own cells and of the next cell along the axis (recomputed from the shared
      // plane, so no R-state exchange and no barrier before the face adjoints), adjoints of the own right (x) and top (y)
      // faces, publish the R-side cotangents
      T* const Bx_s = Rxs + bp * G::XARR;           // [2][5][TY][RXP]  (Rxs, Bxs are contiguous: two buffers)
      T* const By_s = Rys + bp * G::YARR;           // [2][5][TY+1][RTX]
      P2<T> Lbx[5], Lby[5];
      T RbxA[5];                                    // Rb of the face between the two own cells (belongs to the second cell)
      // One copy of the (large) packed adjoint serves both axes: the y pass hands it the state with the components
      // permuted so that the face normal is component 1 (the loop is not unrolled; it keeps the plane-loop body small
      // enough for the instruction cache, see profiles/r01c).
      constexpr int PY[5] = {0, 3, 1, 2, 4};        // field f of a y face goes to slot PY[f]: (rho, vy, vz, vx, P)
#pragma unroll 1
      for (int ax = 0; ax < 2; ++ax) {
        P2<T> Lf[5], Rf[5], lam[5], Lb[5], Rb[5];
        if (ax == 0) {
#pragma unroll
          for (int f = 0; f < 5; ++f) {
            const T* row = Wq_s + f * FP + so;
            const P2<T> W = Wprev[f];
            const T wr = row[2], wr2 = row[3];
            const T d0 = W.x - row[-1], d1 = W.y - W.x, d2 = wr - W.y;
            const P2<T> s = {limit1<T, LIM>(d1, d0), limit1<T, LIM>(d2, d1)};
            park_h<T, LIM>(pkx + f * FS, pkxb + f * FS, P2<T>{d1, d2}, P2<T>{d0, d1});
            Lf[f] = fma2(half, s, W);
            const T Rown = fma_(T(-0.5), s.y, W.y);                         // R state of the second own cell
            const T Rnext = fma_(T(-0.5), limit1<T, LIM>(wr2 - wr, d2), wr);   // R state of the cell right of the pack
            Rf[f] = {Rown, Rnext};
            const T gr = Gq_s[f * FP + so + 2];
            lam[f] = mul2(cx, P2<T>{gq[f].y - gq[f].x, gr - gq[f].y});
          }
        } else {
#pragma unroll
          for (int f = 0; f < 5; ++f) {
            const T* row = Wq_s + f * FP + so;
            const P2<T> W = Wprev[f], Wu = rlds2(row + RSW), Wu2 = rlds2(row + 2 * RSW);
            const P2<T> a = sub2(Wu, W), b = sub2(W, rlds2(row - RSW));
            const P2<T> s = limit2<T, LIM>(a, b);
            park_h<T, LIM>(pky + f * FS, pkyb + f * FS, a, b);
            Lf[PY[f]] = fma2(half, s, W);
            Rf[PY[f]] = fma2(nhalf, limit2<T, LIM>(sub2(Wu2, Wu), a), Wu);  // R state of the row above
            lam[PY[f]] = mul2(cy, sub2(rlds2(Gq_s + f * FP + so + RSW), gq[f]));
          }
        }
        if (RS == 0) hllc_vjp2p<T, 0>(Lf, Rf, c, lam, Lb, Rb); else riemann_vjp2<T, 0, RS>(Lf, Rf, c, lam, Lb, Rb);
        if (ax == 0) {
#pragma unroll
          for (int f = 0; f < 5; ++f) { Lbx[f] = Lb[f]; RbxA[f] = Rb[f].x; Bx_s[f * XF + xo + 1] = Rb[f].y; }
        } else {
#pragma unroll
          for (int f = 0; f < 5; ++f) { Lby[f] = Lb[PY[f]]; rsts2(By_s + f * YF + yo + RTX, Rb[PY[f]]); }
        }
      }
      rcp_async_wait_all();                         // cotangent plane p and the next raw plane have landed
      __syncthreads();
      // ---- phase 3: cell cotangents of plane p-1 for x (with the neighbour terms: lanes exchange their encoded c; the
      // two terms that cross the tile edge are left to the gather kernel, which reads the edge cells' c from Ce) and y
      {
        const bool sty = xy && store_ok;
        const long long os1 = os3 + 2 * (long long)NP;
        // last lane of the row that holds a cell of this tile (beyond it the lanes hold the periodic images of the first
        // cells, so the exchange across it is already the right one)
        const int ll = (min(x0 + RTX, nx) - x0) / 2 - 1;
        const bool edge_l = sty && lane == 0, edge_r = sty && lane == ll;
        const long long oe = (((long long)p.sp0 + zrel0 + it - 4) * ny + wrapr(y0 + r, ny)) * (long long)(2 * p.ntx) + 2 * blockIdx.x;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          P2<T> wx, Px, Mx, wy, Py, My, cey;
          if (LIM == 0) {                                  // one factor k per slope; the y term leaves as one encoded word
            const P2<T> kx = rlds2(pkx + f * FS);
            cell_terms_pm2(Lbx[f], P2<T>{Bx_s[f * XF + xo], RbxA[f]}, kx, wx, Px, Mx);
            cell_terms2(Lby[f], rlds2(By_s + f * YF + yo), rlds2(pky + f * FS), wy, cey);
            Py = {enc_sign(Px.x + Mx.x, kx.x), enc_sign(Px.y + Mx.y, kx.y)};    // (reused below as the encoded c^x of the pack)
          } else {
            P2<T> hxa, hxb, hya, hyb;
            fetch_h<T, LIM>(pkx + f * FS, pkxb + f * FS, hxa, hxb);
            fetch_h<T, LIM>(pky + f * FS, pkyb + f * FS, hya, hyb);
            cell_terms_h2(Lbx[f], P2<T>{Bx_s[f * XF + xo], RbxA[f]}, hxa, hxb, wx, Px, Mx);
            cell_terms_h2(Lby[f], rlds2(By_s + f * YF + yo), hya, hyb, wy, Py, My);
          }
          T pl = shfl_up1(Px.y), mr = shfl_dn1(Mx.x);
          if (lane == 0) pl = T(0);
          if (lane == 31) mr = T(0);
          wx.x += pl - Mx.y;
          wx.y += Px.x - mr;
          rsts2(pk2 + f * FS, add2(wx, wy));
          if (LIM == 0) {                                   // one of P, M is zero: one word with the branch flag in its LSB
            if (sty) rstg2(p.C + f * SPN + os1, cey);
            if (edge_l) p.Ce[f * p.SPE + oe] = Py.x;
            if (edge_r) p.Ce[f * p.SPE + oe + 1] = Py.y;
          } else {                                          // both branches contribute: P and M travel separately
            if (sty) { rstg2(p.C + f * SPN + os1, Py); rstg2(p.C + (5 + f) * SPN + os1, My); }
            if (edge_l) p.Ce[f * p.SPE + oe] = Mx.x;        // what the last cell of the tile on the left loses
            if (edge_r) p.Ce[f * p.SPE + oe + 1] = Px.y;    // what the first cell of the tile on the right receives
          }
        }
      }
      // plane p becomes plane p-1
#pragma unroll
      for (int f = 0; f < 5; ++f) Wprev[f] = rlds2(Wp_s + f * FP + so);
      os3 += (long long)NP;
      op = opn;
      pz = pzn;
    }
  } else {
    // -------------------------------------------------------------------------------------- helper
    constexpr int HP = G::HP, HC = RSW / 2;
    int hg[HP], hs[HP];
#pragma unroll
    for (int k = 0; k < HP; ++k) {
      const int idx = lane + 32 * k;
      int row, cp;
      if (idx < 4 * HC) {
        const int hr = idx / HC;
        cp = idx - hr * HC;
        row = hr < 2 ? hr - 2 : TY + hr - 2;
      } else {
        const int kk = idx - 4 * HC;
        row = kk >> 1;
        cp = (kk & 1) ? HC - 1 : 0;
      }
      hg[k] = (idx < G::NHALO) ? wrapr(y0 + row, ny) * nx + wrapr(x0 - 2 + 2 * cp, nx) : -1;
      hs[k] = (row + 2) * RSW + 2 * cp;
    }
    const int rl = lane < TY ? lane : TY - 1;      // row of the x pass (lanes >= TY repeat the last row, unused)

#pragma unroll 1
    for (int it = 0; it < nit; ++it) {
      const int bp = it & 1, bq = bp ^ 1;
      const T* const Wq_s = Wsm + bq * G::PLANE;
      const T* const Gq_s = Gsm + bq * G::PLANE;
      const size_t op = (size_t)pz * NP;
      // halo of plane p: raw state to registers (converted below), cotangent straight into its shared plane
      P2<T> Uh[HP][5];
#pragma unroll
      for (int k = 0; k < HP; ++k) {
        if (hg[k] >= 0) {
#pragma unroll
          for (int f = 0; f < 5; ++f) {
            Uh[k][f] = rldg2(p.U + f * N + op + hg[k]);
            rcp_async_pack(Gsm + bp * G::PLANE + f * FP + hs[k], p.g + f * N + op + hg[k]);
          }
        }
      }
      rcp_async_commit();
      // the two faces nobody in the tile owns, plane p-1: bottom y face row and left x face column (row rl).  L and R
      // states come from the shared plane of the previous iteration; only the R-side cotangents are needed here.
      T* const Bx_s = Rxs + bp * G::XARR;
      T* const By_s = Rys + bp * G::YARR;
      {
        P2<T> Lf[5], Rf[5], lam[5], Lb[5], Rb[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T* col = Wq_s + f * FP + 2 * lane + 2;
          const P2<T> Wm2 = rlds2(col), Wm1 = rlds2(col + RSW), W0 = rlds2(col + 2 * RSW), W1 = rlds2(col + 3 * RSW);
          const P2<T> d0 = sub2(W0, Wm1);
          Lf[f] = fma2(half, limit2<T, LIM>(d0, sub2(Wm1, Wm2)), Wm1);
          Rf[f] = fma2(nhalf, limit2<T, LIM>(sub2(W1, W0), d0), W0);
          const T* gc = Gq_s + f * FP + 2 * lane + 2;
          lam[f] = mul2(cy, sub2(rlds2(gc + 2 * RSW), rlds2(gc + RSW)));
        }
        riemann_vjp2<T, 1, RS>(Lf, Rf, c, lam, Lb, Rb);   // bottom y face of the tile
#pragma unroll
        for (int f = 0; f < 5; ++f) rsts2(By_s + f * YF + 2 * lane, Rb[f]);
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T* rw = Wq_s + f * FP + (rl + 2) * RSW;
          const T dc = rw[2] - rw[1];
          Lf[f] = bc2(fma_(T(0.5), limit1<T, LIM>(dc, rw[1] - rw[0]), rw[1]));
          Rf[f] = bc2(fma_(T(-0.5), limit1<T, LIM>(rw[3] - rw[2], dc), rw[2]));
          const T* gr = Gq_s + f * FP + (rl + 2) * RSW;
          lam[f] = bc2(p.coef[0] * (gr[2] - gr[1]));
        }
        riemann_vjp2<T, 0, RS>(Lf, Rf, c, lam, Lb, Rb);   // left x face of the tile, row rl
        if (lane < TY) {
#pragma unroll
          for (int f = 0; f < 5; ++f) Bx_s[f * XF + rl * RXP] = Rb[f].x;
        }
      }
      // halo primitives of plane p -> shared
      {
        T* Wb = Wsm + bp * G::PLANE;
#pragma unroll
        for (int k = 0; k < HP; ++k) {
          if (hg[k] >= 0) {
            P2<T> Wh[5];
            prim2(Uh[k], c, Wh);
#pragma unroll
            for (int f = 0; f < 5; ++f) rsts2(Wb + f * FP + hs[k], Wh[f]);
          }
        }
      }
      rcp_async_wait_all();
      __syncthreads();
      ++pz;
      if (pz == nz) pz = 0;
    }
  }
}

// ------------------------------------------------------------------------------------------------ kernel B
// One thread per pack (two x-adjacent cells) of a slab plane: adds the y neighbour terms (rows j -+ 1 of C) and, for the
// packs at a tile edge, the x term that crossed it (Ce), then Ub = prim_vjp(U, Wb) + w1 b1 + w2 b2.
template <class T, int LIM>
__global__ void __launch_bounds__(128, 16) rev_gather_kernel(const RevGatherParams<T> p) {
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;       // pack index along x
  const int i = 2 * ip, j = blockIdx.y, kz = blockIdx.z;      // kz: plane relative to p.z0
  if (i >= p.nx) return;
  const int nx = p.nx, ny = p.ny;
  const size_t NP = (size_t)nx * ny, N = NP * p.nz, SPN = (size_t)p.SP * NP;
  const size_t row = (size_t)j * nx, rowm = (size_t)(j == 0 ? ny - 1 : j - 1) * nx, rowp = (size_t)(j == ny - 1 ? 0 : j + 1) * nx;
  const size_t sp = (size_t)(p.sp0 + kz) * NP;                // scratch plane of this cell
  const size_t cell = (size_t)(p.z0 + kz) * NP + row + i;     // p.z0 + kz < nz by construction
  const int tile = i / RTX, ti = i - tile * RTX;
  const bool el = ti == 0, er = ti == RTX - 2;                // the pack holds the first / last cell of a full tile row
  const int tl = tile == 0 ? p.ntx - 1 : tile - 1, tr = (i + 2 >= nx) ? 0 : tile + 1;
  const size_t oe = ((size_t)(p.sp0 + kz) * ny + j) * (size_t)(2 * p.ntx);
  P2<T> Wb[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    P2<T> w = rldg2(p.Wp + f * SPN + sp + row + i);
    if (LIM == 0) {                                           // encoded c: the flag says which neighbour it belongs to
      const T* Cy = p.C + f * SPN + sp + i;
      const P2<T> cd = rldg2(Cy + rowm), cu = rldg2(Cy + rowp);
      w.x += pterm(cd.x) - mterm(cu.x);
      w.y += pterm(cd.y) - mterm(cu.y);
      if (el) w.x += pterm(p.Ce[f * p.SPE + oe + 2 * tl + 1]);
      if (er) w.y -= mterm(p.Ce[f * p.SPE + oe + 2 * tr]);
    } else {                                                  // P of the row below, M of the row above
      const P2<T> pd = rldg2(p.C + f * SPN + sp + i + rowm), mu = rldg2(p.C + (5 + f) * SPN + sp + i + rowp);
      w.x += pd.x - mu.x;
      w.y += pd.y - mu.y;
      if (el) w.x += p.Ce[f * p.SPE + oe + 2 * tl + 1];
      if (er) w.y -= p.Ce[f * p.SPE + oe + 2 * tr];
    }
    Wb[f] = w;
  }
  P2<T> U[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) U[f] = rldg2(p.U + f * N + cell);
  T u[5], wb[5], ubx[5], uby[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) { u[f] = U[f].x; wb[f] = Wb[f].x; }
  prim_vjp(u, p.c, wb, ubx);
#pragma unroll
  for (int f = 0; f < 5; ++f) { u[f] = U[f].y; wb[f] = Wb[f].y; }
  prim_vjp(u, p.c, wb, uby);
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    P2<T> v = {ubx[f], uby[f]};
    if (p.b1) v = fma2(bc2(p.w1), rldg2(p.b1 + f * N + cell), v);
    if (p.b2) v = fma2(bc2(p.w2), rldg2(p.b2 + f * N + cell), v);
    rstg2(p.out + f * N + cell, v);
  }
}

// ------------------------------------------------------------------------------------------------ launchers
// words of scratch per cell of a slab: Wp 5 + c^y 5 (minmod: one encoded word; van Leer / MC: P and M separately, 10)
int rev_scratch_words(int limiter) { return limiter == 0 ? 10 : 15; }

namespace {
template <class T, int LIM, int RS>
cudaError_t launch_rev_faces_l(const RevFaceParams<T>& p, int sm_count, cudaStream_t s) {
  constexpr int NW = sizeof(T) == 4 ? 8 : 4;      // fp64 (parity only): 3 row warps so that shared memory fits
  using G = GeoR<NW>;
  const size_t smem = (size_t)G::TOTAL * sizeof(T);
  static bool configured[64] = {};    // per device: the attribute belongs to the (function, device) pair
  int cur_dev = 0;
  cudaGetDevice(&cur_dev);
  if (cur_dev < 0 || cur_dev >= 64 || !configured[cur_dev]) {
    cudaError_t e = cudaFuncSetAttribute((const void*)rev_faces_kernel<T, NW, LIM, RS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (cur_dev >= 0 && cur_dev < 64) configured[cur_dev] = true;
  }
  const int bx = (p.nx + RTX - 1) / RTX, by = (p.ny + G::TY - 1) / G::TY;
  // z chunks: waves of sm_count blocks (one block per SM), 6 lead-in / lead-out planes per chunk
  const long long tiles = (long long)bx * by;
  int bz = 1;
  long long best = -1;
  for (int cand = 1; cand <= (p.nout + 3) / 4 && cand <= 65535; ++cand) {
    const int zl_c = (p.nout + cand - 1) / cand;
    if ((p.nout + zl_c - 1) / zl_c != cand) continue;
    const long long cost = ((tiles * cand + sm_count - 1) / sm_count) * (zl_c + 6);
    if (best < 0 || cost < best) { best = cost; bz = cand; }
  }
  const int ZL = (p.nout + bz - 1) / bz;
  dim3 grid(bx, by, bz), block(NW * 32);
  rev_faces_kernel<T, NW, LIM, RS><<<grid, block, smem, s>>>(p, ZL);
  return cudaGetLastError();
}
}  // namespace

template <class T>
cudaError_t launch_rev_faces(const RevFaceParams<T>& p, int limiter, int riemann, int sm_count, cudaStream_t s) {
  switch (limiter * 3 + riemann) {
    case 1: return launch_rev_faces_l<T, 0, 1>(p, sm_count, s);
    case 2: return launch_rev_faces_l<T, 0, 2>(p, sm_count, s);
    case 3: return launch_rev_faces_l<T, 1, 0>(p, sm_count, s);
    case 4: return launch_rev_faces_l<T, 1, 1>(p, sm_count, s);
    case 5: return launch_rev_faces_l<T, 1, 2>(p, sm_count, s);
    case 6: return launch_rev_faces_l<T, 2, 0>(p, sm_count, s);
    case 7: return launch_rev_faces_l<T, 2, 1>(p, sm_count, s);
    case 8: return launch_rev_faces_l<T, 2, 2>(p, sm_count, s);
    default: return launch_rev_faces_l<T, 0, 0>(p, sm_count, s);
  }
}

template <class T>
cudaError_t launch_rev_gather(const RevGatherParams<T>& p, int limiter, cudaStream_t s) {
  dim3 block(128), grid((p.nx / 2 + 127) / 128, p.ny, p.nplanes);
  if (limiter == 0) rev_gather_kernel<T, 0><<<grid, block, 0, s>>>(p);
  else rev_gather_kernel<T, 1><<<grid, block, 0, s>>>(p);
  return cudaGetLastError();
}

template cudaError_t launch_rev_faces<float>(const RevFaceParams<float>&, int, int, int, cudaStream_t);
template cudaError_t launch_rev_faces<double>(const RevFaceParams<double>&, int, int, int, cudaStream_t);
template cudaError_t launch_rev_gather<float>(const RevGatherParams<float>&, int, cudaStream_t);
template cudaError_t launch_rev_gather<double>(const RevGatherParams<double>&, int, cudaStream_t);

}  // namespace dh
