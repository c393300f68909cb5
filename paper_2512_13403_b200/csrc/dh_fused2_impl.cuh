// dh_fused2_impl.cuh — fused z-sweep stage kernel, 2x2 footprint (DH_OPT_KERNEL = 0): steps a2-a6 of SURVEY.md §8(a)
// in one launch per RK2 stage:
//     out = B - tau * sum_a (F_{a,+1/2} - F_{a,-1/2}) / dx_a   (+ cooling),   tau = frac * dt
// (PAPER.md:849 Eq. A4, PAPER.md:862-866 Eqs. A6-A7).
//
// Why this shape (profiles/r01b_*): the first fused kernel (dh_fused.cu: one pack per thread, R
// states and fluxes of both in-plane directions exchanged through shared memory, two block barriers per plane)
// is bound by the SM's shared-memory / L1 data pipe (3.4 wavefronts per cell, 62 % of the pipe at 3.4 ms) and
// by barrier stalls, not by HBM.  Here every thread owns a 2 x 2 patch of the plane (two packs of two x-adjacent
// cells, in rows j and j+1), which removes the y exchange inside the patch, and the remaining exchanges are
// arranged so that ONE block barrier per plane suffices:
//  * z lives in registers (previous plane's primitives, its z difference, the left z face state, the partial
//    update), as before; every z face is computed once;
//  * x: a warp owns 64 cells of two rows.  R states and fluxes cross lanes through a per-warp shared array
//    guarded by __syncwarp only; the tile's left-face flux and the R state right of the tile are supplied by
//    the helper warp one plane ahead (it loads the few columns it needs itself);
//  * y: the face between the thread's two rows is private.  The face above them is computed by the thread
//    (the slope of the row above is recomputed from the shared primitive plane, so no R exchange), and its
//    flux is published for the thread above, which subtracts it one iteration later when it finishes the plane;
//  * the helper warp loads and converts the halo (2 rows below, 2 above, 2 columns left and right), computes
//    the tile's bottom y-face row, the left x-face column and the right R column.
// Periodic wrap is index arithmetic on the loads (any tile may straddle it); ragged tiles load wrapped (valid)
// cells and predicate the stores.  The loop body is branch-free: lead-in / lead-out planes run the same
// instructions on data nobody stores.
// One translation unit per Riemann flux (dh_fused2.cu HLLC, dh_fused2_hll.cu, dh_fused2_rusanov.cu) includes this file
// and instantiates launch_stage_fused2_rs<T, RS, COMBO>; they compile side by side.
#pragma once
#include <cstdio>
#include "dh_internal.cuh"
#include "dh_pack.cuh"

namespace dh {

// -DDH_TIMING_PROBE (DH_BUILD_DEFINES=-DDH_TIMING_PROBE python -m paper_2512_13403_b200.build --force): lane 0 of every warp
// of block (1, 1, 0) prints the SM cycles it spends in plane 40 of its sweep, from the top of the loop body to its arrival
// at the block barrier (profiles/r02d_issue_bound.md).  Compiled out otherwise.
#ifdef DH_TIMING_PROBE
#define DH_PROBE_BEGIN const bool prb_ = blockIdx.x == 1 && blockIdx.y == 1 && blockIdx.z == 0 && it == 40 && lane == 0; long long prb_t0 = 0; if (prb_) prb_t0 = clock64();
#define DH_PROBE_END(tag) if (prb_) printf("probe warp %2d %s start %lld cycles %lld\n", w, tag, prb_t0, clock64() - prb_t0);
#else
#define DH_PROBE_BEGIN
#define DH_PROBE_END(tag)
#endif

namespace {

constexpr int TX2 = 64;        // cells per tile row = 32 lanes x 2
constexpr int SW2 = TX2 + 4;   // row pitch of the shared primitive plane (halo 2 on both sides)
constexpr int XP2 = 34;        // pitch of the per-row x exchange arrays (slots 0..32)

template <int NRW> struct Geo2 {
  static constexpr int TY = 2 * NRW;                       // tile rows
  static constexpr int SR = TY + 4;                        // rows of the shared plane (-2 .. TY+1)
  static constexpr int PLANE = 5 * SR * SW2;               // one primitive plane, all 5 fields
  static constexpr int FY = 5 * (NRW + 1) * TX2;           // top-face y fluxes: slot 0 helper, slot r+1 thread row r
  static constexpr int XE = 5 * TY * XP2;                  // x exchange (R states or fluxes), one slot set per row
  static constexpr int STAGE = 5 * TY * TX2;               // cp.async staging of one raw plane of the tile
  static constexpr int TOTAL = 2 * PLANE + 2 * FY + 4 * XE + 3 * STAGE;
  static constexpr int XPK = (TY * 4 + 31) / 32;           // x-edge packs per helper lane (4 per row)
};

DH_DI int wrapm2(int i, int n) {   // i mod n for any i
  int r = i % n;
  return r < 0 ? r + n : r;
}

template <class T> DH_DI P2<T> lds2_(const T* p) { return *reinterpret_cast<const P2<T>*>(p); }
template <class T> DH_DI void sts2_(T* p, P2<T> v) { *reinterpret_cast<P2<T>*>(p) = v; }
template <class T> DH_DI P2<T> ldg2_(const T* p) { return *reinterpret_cast<const P2<T>*>(p); }
template <class T> DH_DI void stg2_(T* p, P2<T> v) { *reinterpret_cast<P2<T>*>(p) = v; }

template <class T> DH_DI void cp_async_pack2(T* smem_dst, const T* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (sizeof(T) == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
template <class T> DH_DI void cp_async_quad2(T* smem_dst, const T* gmem_src) {   // 4 x fp32: 16 bytes
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
DH_DI void cp_async_commit2() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> DH_DI void cp_async_wait2() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// L (= W + s/2) and R (= W - s/2) states of the two cells of a pack along x; wl / wr are the scalar neighbours
template <class T, int LIM>
DH_DI void recon_x2(P2<T> W, T wl, T wr, P2<T>& L, P2<T>& R) {
  const T d0 = W.x - wl, d1 = W.y - W.x, d2 = wr - W.y;
  const P2<T> s = {limit1s<T, LIM>(d1, d0), limit1s<T, LIM>(d2, d1)};
  L = fma2(bc2(T(0.5) / SlopeScale<T, LIM>::k), s, W);
  R = fma2(bc2(T(-0.5) / SlopeScale<T, LIM>::k), s, W);
}

}  // namespace

template <class T, int LIM, int RS, int NRW, bool V16, bool CAND, bool COMBO>
__global__ void __launch_bounds__((NRW + 1) * 32, 1)
stage_fused2_kernel(const StageParams<T> p, const int ZL) {
  using G = Geo2<NRW>;
  constexpr int TY = G::TY, SR = G::SR, FP = SR * SW2;       // FP: field pitch inside a shared plane
  constexpr int FYP = (NRW + 1) * TX2, XEP = TY * XP2, FS = TY * TX2;   // field pitches of the other arrays
  extern __shared__ __align__(16) unsigned char smem_raw2[];
  T* const Wsm = reinterpret_cast<T*>(smem_raw2);  // [2][5][SR][SW2]     primitive planes p (it&1) and p-1
  T* const Fys = Wsm + 2 * G::PLANE;               // [2][5][NRW+1][TX2]  top-face y flux of thread row r in slot r+1
  T* const Rxs = Fys + 2 * G::FY;                  // [2][5][TY][XP2]     R state of the first cell of lane l; slot 32: helper
  T* const Fxs = Rxs + 2 * G::XE;                  // [2][5][TY][XP2]     x flux through the LEFT face of lane l; slot 0: helper
  T* const Ust = Fxs + 2 * G::XE;                  // [5][TY][TX2]        raw U of the next plane (cp.async, private slots)
  T* const Bst = Ust + G::STAGE;                   // [2][5][TY][TX2]     base state, loaded one plane ahead (cp.async, private slots)
  T* const Xst = Bst + 2 * G::STAGE;               // [2][5][TY][TX2]     raw U of planes p, p-1 (COMBO launches only: they get the room)

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const size_t NP = (size_t)nx * ny, N = NP * nz;
  const int x0 = blockIdx.x * TX2, y0 = blockIdx.y * TY, z0 = p.zbeg + blockIdx.z * ZL;
  const int zl = min(ZL, p.zbeg + p.zcnt - z0);
  const int nit = zl + 4;                          // planes z0-2 .. z0+zl+1
  const T dt = p.dt_dev ? *p.dt_dev : p.dt;
  const T tau = p.frac * dt;
  const P2<T> ncx = bc2(-tau * p.inv_dx[0]);
  const P2<T> cy = bc2(tau * p.inv_dx[1]), ncy = bc2(-tau * p.inv_dx[1]);
  const P2<T> cz = bc2(tau * p.inv_dx[2]), ncz = bc2(-tau * p.inv_dx[2]);
  const P2<T> half = bc2(T(0.5) / SlopeScale<T, LIM>::k), nhalf = bc2(T(-0.5) / SlopeScale<T, LIM>::k);   // of the scaled slopes (limit2s)
  const Consts<T>& c = p.c;
  const T cand_thr = CAND ? p.cand_thr[0] : T(0);   // CAND: push the CFL candidates of the result (dh_advance)
  constexpr bool combo = COMBO;                     // out = wB B + wX U - tau D(U): the base state is formed here
  int pz = wrapm2(z0 - 2, nz);
  size_t op = (size_t)pz * NP, opm1 = op, opm2 = op;   // element offsets of planes p, p-1, p-2

  if (w < NRW) {
    // ------------------------------------------------------------------------------------ row warp
    const int r = w, jA = 2 * r, jB = jA + 1;
    const int xg = wrapm2(x0 + 2 * lane, nx);
    const size_t oA = (size_t)wrapm2(y0 + jA, ny) * nx + xg, oB = (size_t)wrapm2(y0 + jB, ny) * nx + xg;
    const bool okx = (x0 + 2 * lane < nx);
    const bool okA = okx && (y0 + jA < ny), okB = okx && (y0 + jB < ny);
    const int soA = (jA + 2) * SW2 + 2 * lane + 2, soB = soA + SW2;   // own packs inside a shared plane
    const int stA = jA * TX2 + 2 * lane, stB = stA + TX2;             // staging slots
    const int xeA = jA * XP2 + lane, xeB = xeA + XP2;                 // x exchange slots
    P2<T> WA[5], dA[5], LzA[5], accA[5], WB[5], dB[5], LzB[5], accB[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) WA[f] = dA[f] = LzA[f] = accA[f] = WB[f] = dB[f] = LzB[f] = accB[f] = bc2(T(0));
    // V16 (fp32, nx % 4 == 0): a lane pair shares the staging work: the even lane copies the 4 cells of row A that the
    // pair owns, the odd lane those of row B, as ONE 16-byte cp.async each (half the LDGSTS count; a __syncwarp
    // makes the partner's copy visible)
    const int q4 = 4 * (lane >> 1);
    const size_t oQ = (size_t)wrapm2(y0 + jA + (lane & 1), ny) * nx + wrapm2(x0 + q4, nx);
    const int stQ = (jA + (lane & 1)) * TX2 + q4;
    if (V16) {
#pragma unroll
      for (int f = 0; f < 5; ++f) cp_async_quad2(Ust + f * FS + stQ, p.U + f * N + op + oQ);
    } else {
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        cp_async_pack2(Ust + f * FS + stA, p.U + f * N + op + oA);
        cp_async_pack2(Ust + f * FS + stB, p.U + f * N + op + oB);
      }
    }
    cp_async_commit2();

#pragma unroll 1
    for (int it = 0; it < nit; ++it) {
      DH_PROBE_BEGIN
      const int bp = it & 1, bq = bp ^ 1;
      T* const Wp_s = Wsm + bp * G::PLANE;
      const T* const Wq_s = Wsm + bq * G::PLANE;
      cp_async_wait2<0>();
      if (V16) __syncwarp();
      P2<T> NA[5], NB[5];                          // plane p: raw, then primitive
#pragma unroll
      for (int f = 0; f < 5; ++f) { NA[f] = lds2_(Ust + f * FS + stA); NB[f] = lds2_(Ust + f * FS + stB); }
      if (combo) {                                 // kept for the base state of this plane, formed one iteration later
#pragma unroll
        for (int f = 0; f < 5; ++f) { sts2_(Xst + bp * G::STAGE + f * FS + stA, NA[f]); sts2_(Xst + bp * G::STAGE + f * FS + stB, NB[f]); }
      }
      // one plane ahead: the raw state of plane p+1 and the base state of plane p (used in the next iteration)
      int pzn = pz + 1;
      size_t opn = op + NP;
      if (pzn == nz) { pzn = 0; opn = 0; }
      if (V16) {
        __syncwarp();                              // the partner has read its half of the slots written below
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          cp_async_quad2(Ust + f * FS + stQ, p.U + f * N + opn + oQ);
          cp_async_quad2(Bst + bp * G::STAGE + f * FS + stQ, p.B + f * N + op + oQ);
        }
      } else {
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          cp_async_pack2(Ust + f * FS + stA, p.U + f * N + opn + oA);
          cp_async_pack2(Ust + f * FS + stB, p.U + f * N + opn + oB);
          cp_async_pack2(Bst + bp * G::STAGE + f * FS + stA, p.B + f * N + op + oA);
          cp_async_pack2(Bst + bp * G::STAGE + f * FS + stB, p.B + f * N + op + oB);
        }
      }
      cp_async_commit2();
      {
        P2<T> t[5];
        prim2(NA, c, t);
#pragma unroll
        for (int f = 0; f < 5; ++f) { NA[f] = t[f]; sts2_(Wp_s + f * FP + soA, t[f]); }
        prim2(NB, c, t);
#pragma unroll
        for (int f = 0; f < 5; ++f) { NB[f] = t[f]; sts2_(Wp_s + f * FP + soB, t[f]); }
      }
      // the bottom y flux of plane p-2 (published by the thread row below in the previous iteration)
#pragma unroll
      for (int f = 0; f < 5; ++f) accA[f] = fma2(cy, lds2_(Fys + bq * G::FY + f * FYP + r * TX2 + 2 * lane), accA[f]);

      // ---- z: slope of plane p-1, face between p-2 and p-1; its flux finishes plane p-2 and opens plane p-1
      const bool st = (it >= 4);
#define DH_ZPHASE(N_, W_, d_, Lz_, acc_, ok_, o_, st_)                                              \
      {                                                                                             \
        P2<T> Rz[5], Fz[5], s[5];                                                                   \
        _Pragma("unroll") for (int f = 0; f < 5; ++f) {                                             \
          const P2<T> a = sub2(N_[f], W_[f]);                                                       \
          s[f] = limit2s<T, LIM>(a, d_[f]);                                                          \
          Rz[f] = fma2(nhalf, s[f], W_[f]);                                                         \
          d_[f] = a;                                                                                \
        }                                                                                           \
        riemann2<T, 2, RS>(Lz_, Rz, c, Fz);                                                                \
        _Pragma("unroll") for (int f = 0; f < 5; ++f) Lz_[f] = fma2(half, s[f], W_[f]);             \
        P2<T> Uo[5];                                                                                \
        _Pragma("unroll") for (int f = 0; f < 5; ++f) Uo[f] = fma2(ncz, Fz[f], acc_[f]);            \
        if (p.cool) cool2(Uo, dt, c);                                                               \
        if (st && ok_) {                                                                            \
          _Pragma("unroll") for (int f = 0; f < 5; ++f) stg2_(p.out + f * N + opm2 + o_, Uo[f]);    \
          if (CAND && cfl_candidate2(Uo, c, cand_thr)) {                                           \
            const unsigned slot = atomicAdd(p.cand_cnt, 1u);                                        \
            if (slot < p.cand_cap) p.cand_list[slot] = (unsigned)(opm2 + o_);                       \
          }                                                                                         \
        }                                                                                           \
        _Pragma("unroll") for (int f = 0; f < 5; ++f) {                                             \
          P2<T> b = lds2_(Bst + bq * G::STAGE + f * FS + st_);                                      \
          if (combo) b = fma2(bc2(p.wX), lds2_(Xst + bq * G::STAGE + f * FS + st_), mul2(bc2(p.wB), b)); \
          acc_[f] = fma2(cz, Fz[f], b);                                                             \
        }                                                                                           \
      }
      DH_ZPHASE(NA, WA, dA, LzA, accA, okA, oA, stA)
      // x neighbours of plane p-1, loaded here so that their latency hides behind the second z phase
      T xl[5][2], xr[5][2];
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        const T* rowA = Wq_s + f * FP + soA;
        xl[f][0] = rowA[-1]; xr[f][0] = rowA[2]; xl[f][1] = rowA[SW2 - 1]; xr[f][1] = rowA[SW2 + 2];
      }
      DH_ZPHASE(NB, WB, dB, LzB, accB, okB, oB, stB)
#undef DH_ZPHASE

      // ---- x on plane p-1 (centre W?): lanes exchange R states and fluxes through per-row slots
      {
        T* const Rx_s = Rxs + bq * G::XE;
        T* const Fx_s = Fxs + bq * G::XE;
        P2<T> LxA[5], RxA[5], LxB[5], RxB[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          recon_x2<T, LIM>(WA[f], xl[f][0], xr[f][0], LxA[f], RxA[f]);
          recon_x2<T, LIM>(WB[f], xl[f][1], xr[f][1], LxB[f], RxB[f]);
          Rx_s[f * XEP + xeA] = RxA[f].x;
          Rx_s[f * XEP + xeB] = RxB[f].x;
        }
        __syncwarp();
        P2<T> FA[5], FB[5];
        {
          P2<T> Rf[5];
#pragma unroll
          for (int f = 0; f < 5; ++f) Rf[f] = {RxA[f].y, Rx_s[f * XEP + xeA + 1]};
          riemann2<T, 0, RS>(LxA, Rf, c, FA);
#pragma unroll
          for (int f = 0; f < 5; ++f) Rf[f] = {RxB[f].y, Rx_s[f * XEP + xeB + 1]};
          riemann2<T, 0, RS>(LxB, Rf, c, FB);
        }
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          Fx_s[f * XEP + xeA + 1] = FA[f].y;
          Fx_s[f * XEP + xeB + 1] = FB[f].y;
        }
        __syncwarp();
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T flA = Fx_s[f * XEP + xeA], flB = Fx_s[f * XEP + xeB];
          const P2<T> dFA = {FA[f].x - flA, FA[f].y - FA[f].x}, dFB = {FB[f].x - flB, FB[f].y - FB[f].x};
          accA[f] = fma2(ncx, dFA, accA[f]);
          accB[f] = fma2(ncx, dFB, accB[f]);
        }
      }
      // ---- y on plane p-1: private face between the two rows, and the face above them (published)
      {
        P2<T> L1[5], R1[5], L2[5], R2[5], F1[5], F2[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T* col = Wq_s + f * FP + soA;
          const P2<T> Wm = lds2_(col - SW2), W2 = lds2_(col + 2 * SW2), W3 = lds2_(col + 3 * SW2);
          const P2<T> dBA = sub2(WB[f], WA[f]), d2B = sub2(W2, WB[f]);
          const P2<T> sA = limit2s<T, LIM>(dBA, sub2(WA[f], Wm));
          const P2<T> sB = limit2s<T, LIM>(d2B, dBA);
          const P2<T> s2 = limit2s<T, LIM>(sub2(W3, W2), d2B);
          L1[f] = fma2(half, sA, WA[f]);
          R1[f] = fma2(nhalf, sB, WB[f]);
          L2[f] = fma2(half, sB, WB[f]);
          R2[f] = fma2(nhalf, s2, W2);
        }
        riemann2<T, 1, RS>(L1, R1, c, F1);
        riemann2<T, 1, RS>(L2, R2, c, F2);
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          sts2_(Fys + bp * G::FY + f * FYP + (r + 1) * TX2 + 2 * lane, F2[f]);
          accA[f] = fma2(ncy, F1[f], accA[f]);           // its bottom flux arrives in the next iteration
          accB[f] = fma2(cy, F1[f], fma2(ncy, F2[f], accB[f]));
        }
      }
      // plane p becomes plane p-1
#pragma unroll
      for (int f = 0; f < 5; ++f) { WA[f] = NA[f]; WB[f] = NB[f]; }
      opm2 = opm1;
      opm1 = op;
      op = opn;
      pz = pzn;
      DH_PROBE_END("row")
      __syncthreads();
    }
  } else {
    // -------------------------------------------------------------------------------------- helper
    constexpr int XPK = G::XPK;
    // y halo: pack `lane` of rows -2, -1, TY, TY+1
    const int xg = wrapm2(x0 + 2 * lane, nx);
    size_t hy_g[4];
    int hy_s[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int row = (k < 2) ? k - 2 : TY + k - 2;
      hy_g[k] = (size_t)wrapm2(y0 + row, ny) * nx + xg;
      hy_s[k] = (row + 2) * SW2 + 2 * lane + 2;
    }
    // x edge: pack e = lane + 32 m of row e / 4; kind e % 4: columns {-2,-1}, {0,1}, {62,63}, {64,65}
    size_t hx_g[XPK];
    int hx_s[XPK], hx_row[XPK];
    const int kind = lane & 3;
#pragma unroll
    for (int m = 0; m < XPK; ++m) {
      const int e = lane + 32 * m, row = e >> 2;
      const int col = (kind == 0) ? -2 : (kind == 1) ? 0 : (kind == 2) ? TX2 - 2 : TX2;
      hx_row[m] = (row < TY) ? row : -1;
      hx_g[m] = (size_t)wrapm2(y0 + (row < TY ? row : 0), ny) * nx + wrapm2(x0 + col, nx);
      hx_s[m] = (row + 2) * SW2 + col + 2;
    }

#pragma unroll 1
    for (int it = 0; it < nit; ++it) {
      DH_PROBE_BEGIN
      const int bp = it & 1, bq = bp ^ 1;
      T* const Wp_s = Wsm + bp * G::PLANE;
      const T* const Wq_s = Wsm + bq * G::PLANE;
      // raw halo cells of plane p (consumed after the flux work below, so the loads have time to land)
      P2<T> Uy[4][5], Ux[XPK][5];
#pragma unroll
      for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int f = 0; f < 5; ++f) Uy[k][f] = ldg2_(p.U + f * N + op + hy_g[k]);
#pragma unroll
      for (int m = 0; m < XPK; ++m)
#pragma unroll
        for (int f = 0; f < 5; ++f) Ux[m][f] = ldg2_(p.U + f * N + op + hx_g[m]);
      // bottom y face row of the tile, plane p-1: rows -2 .. 1 of the shared plane
      {
        P2<T> L[5], R[5], F[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T* col = Wq_s + f * FP + 2 * lane + 2;
          const P2<T> Wm2 = lds2_(col), Wm1 = lds2_(col + SW2), W0 = lds2_(col + 2 * SW2), W1 = lds2_(col + 3 * SW2);
          const P2<T> d0 = sub2(W0, Wm1);
          const P2<T> sm = limit2s<T, LIM>(d0, sub2(Wm1, Wm2));
          const P2<T> s0 = limit2s<T, LIM>(sub2(W1, W0), d0);
          L[f] = fma2(half, sm, Wm1);
          R[f] = fma2(nhalf, s0, W0);
        }
        riemann2<T, 1, RS>(L, R, c, F);
#pragma unroll
        for (int f = 0; f < 5; ++f) sts2_(Fys + bp * G::FY + f * FYP + 2 * lane, F[f]);
      }
      // y halo primitives of plane p -> shared
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        P2<T> Wh[5];
        prim2(Uy[k], c, Wh);
#pragma unroll
        for (int f = 0; f < 5; ++f) sts2_(Wp_s + f * FP + hy_s[k], Wh[f]);
      }
      // x edge of plane p: halo columns -> shared; left-face flux (lane kind 0) and right R state (lane kind 3)
#pragma unroll
      for (int m = 0; m < XPK; ++m) {
        P2<T> Wh[5], L[5], R[5], F[5];
        prim2(Ux[m], c, Wh);
        const bool live = hx_row[m] >= 0;
        if (live && (kind == 0 || kind == 3)) {
#pragma unroll
          for (int f = 0; f < 5; ++f) sts2_(Wp_s + f * FP + hx_s[m], Wh[f]);
        }
        T Re[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          // kind 0 holds (W_-2, W_-1) and takes (W_0, W_1) from lane+1; kind 3 holds (W_64, W_65) and takes W_63 from lane-1
          const T nx_ = __shfl_down_sync(0xffffffffu, Wh[f].x, 1), ny_ = __shfl_down_sync(0xffffffffu, Wh[f].y, 1);
          const T pv_ = __shfl_up_sync(0xffffffffu, Wh[f].y, 1);
          const T dl = Wh[f].y - Wh[f].x, dc = nx_ - Wh[f].y, dr = ny_ - nx_;
          const T sl = limit1s<T, LIM>(dc, dl), sc = limit1s<T, LIM>(dr, dc);
          L[f] = bc2(fma_(T(0.5) / SlopeScale<T, LIM>::k, sl, Wh[f].y));
          R[f] = bc2(fma_(T(-0.5) / SlopeScale<T, LIM>::k, sc, nx_));
          const T se = limit1s<T, LIM>(dl, Wh[f].x - pv_);
          Re[f] = fma_(T(-0.5) / SlopeScale<T, LIM>::k, se, Wh[f].x);
        }
        riemann2<T, 0, RS>(L, R, c, F);
        if (live && kind == 0) {
#pragma unroll
          for (int f = 0; f < 5; ++f) Fxs[bp * G::XE + f * XEP + hx_row[m] * XP2] = F[f].x;
        }
        if (live && kind == 3) {
#pragma unroll
          for (int f = 0; f < 5; ++f) Rxs[bp * G::XE + f * XEP + hx_row[m] * XP2 + 32] = Re[f];
        }
      }
      int pzn = pz + 1;
      size_t opn = op + NP;
      if (pzn == nz) { pzn = 0; opn = 0; }
      op = opn;
      pz = pzn;
      DH_PROBE_END("helper")
      __syncthreads();
    }
  }
}

namespace {

template <class T, int LIM, int RS, int NRW, bool V16, bool CAND, bool COMBO>
cudaError_t launch_one2c(const StageParams<T>& p, int sm_count, cudaStream_t s) {
  using G = Geo2<NRW>;
  const size_t smem = (size_t)(G::TOTAL + (COMBO ? 2 * G::STAGE : 0)) * sizeof(T);
  static bool configured[64] = {};    // per instantiation and per device: the attribute belongs to the (function, device) pair
  int cur_dev = 0;
  cudaGetDevice(&cur_dev);
  if (cur_dev < 0 || cur_dev >= 64 || !configured[cur_dev]) {
    cudaError_t e = cudaFuncSetAttribute((const void*)stage_fused2_kernel<T, LIM, RS, NRW, V16, CAND, COMBO>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (cur_dev >= 0 && cur_dev < 64) configured[cur_dev] = true;
  }
  const int bx = (p.nx + TX2 - 1) / TX2, by = (p.ny + G::TY - 1) / G::TY;
  // z chunks: every chunk pays 4 lead-in planes, and blocks run in waves of (blocks per SM) x sm_count;
  // pick the chunk count that minimises waves x (planes per chunk + 4)
  int dev = 0, per_sm = 1;
  cudaGetDevice(&dev);
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, stage_fused2_kernel<T, LIM, RS, NRW, V16, CAND, COMBO>, (NRW + 1) * 32, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
  const long long slots = (long long)per_sm * sm_count, tiles = (long long)bx * by;
  int bz = 1;
  long long best = -1;
  const int zc = p.zcnt;                           // planes of this launch (the whole grid or a z range)
  for (int cand = 1; cand <= (zc < 4 ? 1 : zc / 4) && cand <= 65535; ++cand) {
    const int zl_c = (zc + cand - 1) / cand;
    if ((zc + zl_c - 1) / zl_c != cand) continue;
    const long long cost = ((tiles * cand + slots - 1) / slots) * (zl_c + 4);
    if (best < 0 || cost < best) { best = cost; bz = cand; }
  }
  const int ZL = (zc + bz - 1) / bz;
  dim3 grid(bx, by, bz), block((NRW + 1) * 32);
  stage_fused2_kernel<T, LIM, RS, NRW, V16, CAND, COMBO><<<grid, block, smem, s>>>(p, ZL);
  return cudaGetLastError();
}

template <class T, int LIM, int RS, int NRW, bool V16, bool COMBO>
cudaError_t launch_one2(const StageParams<T>& p, int sm_count, cudaStream_t s) {
  return p.cand_list ? launch_one2c<T, LIM, RS, NRW, V16, true, COMBO>(p, sm_count, s) : launch_one2c<T, LIM, RS, NRW, V16, false, COMBO>(p, sm_count, s);
}

}  // namespace

// COMBO (StageParams::combo, the Shu-Osher stages of Heun / SSPRK3) is a set of instantiations of its own, built in translation
// units of its own (dh_fused2_combo*.cu): a run-time flag costs the default kernel 8 registers and 3-4 %.
template <class T, int RS, bool COMBO>
cudaError_t launch_stage_fused2_rs(const StageParams<T>& p, int limiter, int sm_count, cudaStream_t s, bool* supported) {
  // packs are two cells adjacent in x: nx must be even; grid.y/z <= 65535
  *supported = (p.nx % 2 == 0) && ((p.ny + 5) / 6 <= 65535);
  if (!*supported) return cudaSuccess;
  // fp32: 7 row warps + helper, one block per SM with the full register file (the kernel is bound by issue and
  // register pressure, not occupancy: profiles/r01c); fp64 (parity only): 3 row warps so that shared memory fits
  constexpr int NRW = sizeof(T) == 4 ? 7 : 3;
  if (sizeof(T) == 4 && p.nx % 4 == 0) {             // 16-byte staging copies
    switch (limiter) {
      case 1: return launch_one2<T, 1, RS, NRW, true, COMBO>(p, sm_count, s);
      case 2: return launch_one2<T, 2, RS, NRW, true, COMBO>(p, sm_count, s);
      default: return launch_one2<T, 0, RS, NRW, true, COMBO>(p, sm_count, s);
    }
  }
  if constexpr (COMBO && sizeof(T) == 4) {
    return cudaErrorInvalidValue;                    // combo_ok() in dh_api.cu never asks: fp32 COMBO is built for nx % 4 == 0 only
  } else {
    switch (limiter) {
      case 1: return launch_one2<T, 1, RS, NRW, false, COMBO>(p, sm_count, s);
      case 2: return launch_one2<T, 2, RS, NRW, false, COMBO>(p, sm_count, s);
      default: return launch_one2<T, 0, RS, NRW, false, COMBO>(p, sm_count, s);
    }
  }
}

}  // namespace dh
