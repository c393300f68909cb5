// dh_fused.cu — fused z-sweep stage kernel (DH_OPT_KERNEL = 0): steps a2-a6 of SURVEY.md §8(a) in one launch
// per RK2 stage:   out = B - tau * sum_a (F_{a,+1/2} - F_{a,-1/2}) / dx_a   (+ cooling),  tau = frac * dt
// (PAPER.md:849 Eq. A4, PAPER.md:862-866 Eqs. A6-A7).
//
// Layout of the work ("Kernels"):
//  * a block owns an x-y tile of TX = 64 by TY = NW-1 cells and sweeps ZL planes in z.  Warp r < TY is the
//    "row warp" of tile row r; each of its lanes owns TWO cells adjacent in x (a pack, dh_pack.cuh), so global
//    loads and stores are 8-byte, fully coalesced, and fp32 add/mul/fma issue as FADD2/FMUL2/FFMA2.
//  * the z direction lives in registers: W of the previous plane, its z difference, the left z face state and
//    the partial update of the previous plane are carried from plane to plane; every z face is computed once.
//  * the x and y directions exchange through shared memory: the primitive plane (with a halo of 2) is double
//    buffered; each thread computes the slopes of its own cells, publishes its R states, computes the HLLC flux
//    of its OWN right (x) and top (y) face, publishes it, and reads its left / bottom neighbour's.  Every face
//    of the tile is therefore computed exactly once.
//  * the last warp is the "helper": it loads and converts the halo cells of the plane, and computes the faces
//    nobody owns (the tile's bottom y face row and left x face column) plus the R states of the halo row /
//    column on the other side.
//  * two __syncthreads per plane.  Periodic wrap is index arithmetic on the loads (any tile may straddle it);
//    ragged tiles load wrapped (valid) cells and predicate the stores.
#include "dh_internal.cuh"
#include "dh_pack.cuh"

namespace dh {

namespace {

constexpr int TX = 64;        // cells per tile row = 32 lanes x 2
constexpr int SW = TX + 4;    // row pitch of the shared primitive plane (halo 2 on both sides)
constexpr int XP = 34;        // pitch of the x exchange arrays (33 used)

template <int NW> struct Geo {
  static constexpr int TY = NW - 1;
  static constexpr int SR = TY + 4;                       // rows of the shared plane
  static constexpr int PLANE = 5 * SR * SW;               // one buffered primitive plane (all 5 fields)
  static constexpr int XARR = 5 * TY * XP;
  static constexpr int YARR = 5 * (TY + 1) * TX;
  static constexpr int STAGE = 5 * TY * TX;                // cp.async staging of one raw row-warp plane (all 5 fields)
  static constexpr int TOTAL = 2 * PLANE + 2 * XARR + 2 * YARR + 2 * STAGE;
  static constexpr int NHALO = 4 * (SW / 2) + 2 * TY;     // halo packs per plane
  static constexpr int HP = (NHALO + 31) / 32;            // halo packs per helper lane
};

DH_DI int wrapm(int i, int n) {   // i mod n for any i
  int r = i % n;
  return r < 0 ? r + n : r;
}

template <class T> DH_DI P2<T> lds2(const T* p) { return *reinterpret_cast<const P2<T>*>(p); }
template <class T> DH_DI void sts2(T* p, P2<T> v) { *reinterpret_cast<P2<T>*>(p) = v; }
template <class T> DH_DI P2<T> ldg2(const T* p) { return *reinterpret_cast<const P2<T>*>(p); }
template <class T> DH_DI void stg2(T* p, P2<T> v) { *reinterpret_cast<P2<T>*>(p) = v; }

// 8-byte (fp32 pack) / 16-byte (fp64 pack) asynchronous global -> shared copy of one pack (LDGSTS)
template <class T> DH_DI void cp_async_pack(T* smem_dst, const T* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (sizeof(T) == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
DH_DI void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> DH_DI void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// slopes of the two cells of a pack along x from the scalar neighbours wl (left of .x) and wr (right of .y);
// returns the L (= W + s/2) and R (= W - s/2) states of both cells
template <class T, int LIM>
DH_DI void recon_x(P2<T> W, T wl, T wr, P2<T>& L, P2<T>& R) {
  const T d0 = W.x - wl, d1 = W.y - W.x, d2 = wr - W.y;
  const P2<T> s = {limit1<T, LIM>(d1, d0), limit1<T, LIM>(d2, d1)};
  L = fma2(bc2(T(0.5)), s, W);
  R = fma2(bc2(T(-0.5)), s, W);
}

// slopes along y or z from the packs below (Wm) and above (Wp)
template <class T, int LIM>
DH_DI void recon_p(P2<T> Wm, P2<T> W, P2<T> Wp, P2<T>& L, P2<T>& R) {
  const P2<T> s = limit2<T, LIM>(sub2(Wp, W), sub2(W, Wm));
  L = fma2(bc2(T(0.5)), s, W);
  R = fma2(bc2(T(-0.5)), s, W);
}

}  // namespace

template <class T, int LIM, int NW>
__global__ void __launch_bounds__(NW * 32, (sizeof(T) == 4 && NW <= 8) ? 2 : 1)
stage_fused_kernel(const StageParams<T> p, const int ZL) {
  using G = Geo<NW>;
  constexpr int TY = G::TY, SR = G::SR;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* const Wsm = reinterpret_cast<T*>(smem_raw);   // [2][5][SR][SW]  primitive planes p (it&1) and p-1
  T* const Rxs = Wsm + 2 * G::PLANE;               // [5][TY][XP]     R state of the first cell of lane l (l = 32: halo column)
  T* const Fxs = Rxs + G::XARR;                    // [5][TY][XP]     x flux through the LEFT face of lane l's pack
  T* const Rys = Fxs + G::XARR;                    // [5][TY+1][TX]   R states of row r (r = TY: halo row)
  T* const Fys = Rys + G::YARR;                    // [5][TY+1][TX]   y flux through the BOTTOM face of row r
  T* const Ust = Fys + G::YARR;                    // [5][TY][TX]     raw U of the next plane (cp.async, private per thread)
  T* const Bst = Ust + G::STAGE;                   // [5][TY][TX]     base state of plane p-1 (cp.async, private per thread)

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const size_t NP = (size_t)nx * ny, N = NP * nz;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * ZL;
  const int zl = min(ZL, nz - z0);
  const int nit = zl + 4;                          // planes z0-2 .. z0+zl+1
  const T dt = p.dt_dev ? *p.dt_dev : p.dt;
  const T tau = p.frac * dt;
  const P2<T> ncx = bc2(-tau * p.inv_dx[0]), ncy = bc2(-tau * p.inv_dx[1]);
  const P2<T> cz = bc2(tau * p.inv_dx[2]), ncz = bc2(-tau * p.inv_dx[2]);
  const P2<T> half = bc2(T(0.5)), nhalf = bc2(T(-0.5));
  const Consts<T>& c = p.c;

  if (w < TY) {
    // ------------------------------------------------------------------------------------ row warp
    const int r = w;
    const size_t o = (size_t)wrapm(y0 + r, ny) * nx + wrapm(x0 + 2 * lane, nx);
    const bool store_ok = (x0 + 2 * lane < nx) && (y0 + r < ny);
    const int so = (r + 2) * SW + 2 * lane + 2;    // own pack inside a shared plane
    const int xo = r * XP + lane, yo = r * TX + 2 * lane;
    T* const ust = Ust + yo;                       // this thread's staging slots (stride TY*TX per field)
    T* const bst = Bst + yo;
    constexpr int FS = TY * TX;
    P2<T> Wprev[5], dprev[5], WLz[5], acc[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) Wprev[f] = dprev[f] = WLz[f] = acc[f] = bc2(T(0));
    // element offsets of this thread's pack in planes p, p-1, p-2 (64-bit: 5 N words may exceed 2^32 bytes)
    int pz = wrapm(z0 - 2, nz);
    size_t op = (size_t)pz * NP + o, opm1 = op, opm2 = op;
#pragma unroll
    for (int f = 0; f < 5; ++f) cp_async_pack(ust + f * FS, p.U + f * N + op);
    cp_async_commit();

#pragma unroll 1
    for (int it = 0; it < nit; ++it) {
      const bool xy = (it >= 3) && (it <= zl + 2);   // x/y work on plane p-1 = z0 + it - 3
      cp_async_wait<0>();
      P2<T> Uc[5];
#pragma unroll
      for (int f = 0; f < 5; ++f) Uc[f] = lds2(ust + f * FS);
      // base state of plane p-1 first (needed in this iteration), then the raw state of plane p+1
      if (xy) {
#pragma unroll
        for (int f = 0; f < 5; ++f) cp_async_pack(bst + f * FS, p.B + f * N + opm1);
      }
      cp_async_commit();
      int pzn = pz + 1;
      size_t opn = op + NP;
      if (pzn == nz) { pzn = 0; opn = o; }
      if (it + 1 < nit) {
#pragma unroll
        for (int f = 0; f < 5; ++f) cp_async_pack(ust + f * FS, p.U + f * N + opn);
      }
      cp_async_commit();
      // primitives of plane p -> shared (read by the neighbours in the next iteration)
      P2<T> Wp[5];
      prim2(Uc, c, Wp);
      {
        T* Wb = Wsm + (it & 1) * G::PLANE + so;
#pragma unroll
        for (int f = 0; f < 5; ++f) sts2(Wb + f * SR * SW, Wp[f]);
      }
      // z: slope of cell p-1, face between p-2 and p-1; the face flux finishes plane p-2 and opens plane p-1
      {
        P2<T> Rz[5], Fz[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const P2<T> a = sub2(Wp[f], Wprev[f]);
          const P2<T> s = limit2<T, LIM>(a, dprev[f]);
          Rz[f] = fma2(nhalf, s, Wprev[f]);
          dprev[f] = a;
          Wp[f] = fma2(half, s, Wprev[f]);         // left state of the NEXT z face (kept in WLz below)
        }
        if (it >= 3) hllc2<T, 2>(WLz, Rz, c, Fz);
#pragma unroll
        for (int f = 0; f < 5; ++f) WLz[f] = Wp[f];
        if (it >= 4) {
          P2<T> Uo[5];
#pragma unroll
          for (int f = 0; f < 5; ++f) Uo[f] = fma2(ncz, Fz[f], acc[f]);
          if (p.cool) cool2(Uo, dt, c);
          if (store_ok) {
#pragma unroll
            for (int f = 0; f < 5; ++f) stg2(p.out + f * N + opm2, Uo[f]);
          }
        }
        if (xy) {
          cp_async_wait<1>();                      // the base-state group; the next-plane group may still fly
#pragma unroll
          for (int f = 0; f < 5; ++f) acc[f] = fma2(cz, Fz[f], lds2(bst + f * FS));
        }
      }
      // the primitives of plane p were overwritten above: reload them (own smem slot, no hazard)
      const T* Wq = Wsm + ((it - 1) & 1) * G::PLANE + so;
      // x / y, phase 1: slopes of the own cells of plane p-1, publish the R states
      P2<T> Lx[5], Rxo[5], Ly[5];
      if (xy) {
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T* row = Wq + f * SR * SW;
          recon_x<T, LIM>(Wprev[f], row[-1], row[2], Lx[f], Rxo[f]);
          Rxs[f * TY * XP + xo] = Rxo[f].x;
          P2<T> Ryo;
          recon_p<T, LIM>(lds2(row - SW), Wprev[f], lds2(row + SW), Ly[f], Ryo);
          sts2(Rys + f * (TY + 1) * TX + yo, Ryo);
        }
      }
      __syncthreads();
      // phase 2: HLLC flux through the own right (x) and top (y) faces, publish them
      P2<T> Fx[5], Fy[5];
      if (xy) {
        P2<T> Rf[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) Rf[f] = {Rxo[f].y, Rxs[f * TY * XP + xo + 1]};
        hllc2<T, 0>(Lx, Rf, c, Fx);
#pragma unroll
        for (int f = 0; f < 5; ++f) Fxs[f * TY * XP + xo + 1] = Fx[f].y;
#pragma unroll
        for (int f = 0; f < 5; ++f) Rf[f] = lds2(Rys + f * (TY + 1) * TX + yo + TX);
        hllc2<T, 1>(Ly, Rf, c, Fy);
#pragma unroll
        for (int f = 0; f < 5; ++f) sts2(Fys + f * (TY + 1) * TX + yo + TX, Fy[f]);
      }
      __syncthreads();
      // phase 3: x and y differences into the partial update of plane p-1
      if (xy) {
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T fl = Fxs[f * TY * XP + xo];
          const P2<T> dFx = {Fx[f].x - fl, Fx[f].y - Fx[f].x};
          const P2<T> Fb = lds2(Fys + f * (TY + 1) * TX + yo);
          acc[f] = fma2(ncy, sub2(Fy[f], Fb), fma2(ncx, dFx, acc[f]));
        }
      }
      // plane p becomes plane p-1
      {
        const T* Wn = Wsm + (it & 1) * G::PLANE + so;
#pragma unroll
        for (int f = 0; f < 5; ++f) Wprev[f] = lds2(Wn + f * SR * SW);
      }
      opm2 = opm1;
      opm1 = op;
      op = opn;
      pz = pzn;
    }
  } else {
    // -------------------------------------------------------------------------------------- helper
    constexpr int HP = G::HP, HC = SW / 2;
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
      hg[k] = (idx < G::NHALO) ? wrapm(y0 + row, ny) * nx + wrapm(x0 - 2 + 2 * cp, nx) : -1;
      hs[k] = (row + 2) * SW + 2 * cp;
    }
    const int rl = lane < TY ? lane : TY - 1;      // row of the x pass (lanes >= TY repeat the last row, unused)
    int pz = wrapm(z0 - 2, nz);

#pragma unroll 1
    for (int it = 0; it < nit; ++it) {
      const bool xy = (it >= 3) && (it <= zl + 2);
      // raw halo cells of plane p (consumed after the flux work below, so the loads have time to land)
      P2<T> Uh[HP][5];
#pragma unroll
      for (int k = 0; k < HP; ++k) {
        if (hg[k] >= 0) {
#pragma unroll
          for (int f = 0; f < 5; ++f) Uh[k][f] = ldg2(p.U + f * N + pz * NP + hg[k]);
        }
      }
      P2<T> LyB[5];
      T LxB[5];
      if (xy) {
        const T* Wq = Wsm + ((it - 1) & 1) * G::PLANE;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const T* pl = Wq + f * SR * SW;
          // y: R state of the halo row TY, L state of the halo row -1
          const T* col = pl + 2 * lane + 2;
          P2<T> Lt, Rt;
          recon_p<T, LIM>(lds2(col + (TY + 1) * SW), lds2(col + (TY + 2) * SW), lds2(col + (TY + 3) * SW), Lt, Rt);
          sts2(Rys + f * (TY + 1) * TX + TY * TX + 2 * lane, Rt);
          recon_p<T, LIM>(lds2(col), lds2(col + SW), lds2(col + 2 * SW), LyB[f], Rt);
          // x: L state of the halo column -1, R state of the halo column TX, row rl
          const T* rw = pl + (rl + 2) * SW;
          const T sl = limit1<T, LIM>(rw[2] - rw[1], rw[1] - rw[0]);
          LxB[f] = fma(T(0.5), sl, rw[1]);
          const T sr = limit1<T, LIM>(rw[TX + 3] - rw[TX + 2], rw[TX + 2] - rw[TX + 1]);
          if (lane < TY) Rxs[f * TY * XP + rl * XP + 32] = fma(T(-0.5), sr, rw[TX + 2]);
        }
      }
      __syncthreads();
      if (xy) {
        P2<T> Lf[5], Rf[5], F[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) Rf[f] = lds2(Rys + f * (TY + 1) * TX + 2 * lane);
        hllc2<T, 1>(LyB, Rf, c, F);                 // bottom y face of the tile
#pragma unroll
        for (int f = 0; f < 5; ++f) sts2(Fys + f * (TY + 1) * TX + 2 * lane, F[f]);
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          Lf[f] = bc2(LxB[f]);
          Rf[f] = bc2(Rxs[f * TY * XP + rl * XP]);
        }
        hllc2<T, 0>(Lf, Rf, c, F);                  // left x face of the tile, row rl
        if (lane < TY) {
#pragma unroll
          for (int f = 0; f < 5; ++f) Fxs[f * TY * XP + rl * XP] = F[f].x;
        }
      }
      // halo primitives of plane p -> shared
      {
        T* Wb = Wsm + (it & 1) * G::PLANE;
#pragma unroll
        for (int k = 0; k < HP; ++k) {
          if (hg[k] >= 0) {
            P2<T> Wh[5];
            prim2(Uh[k], c, Wh);
#pragma unroll
            for (int f = 0; f < 5; ++f) sts2(Wb + f * SR * SW + hs[k], Wh[f]);
          }
        }
      }
      __syncthreads();
      ++pz;
      if (pz == nz) pz = 0;
    }
  }
}

namespace {

template <class T, int LIM, int NW>
cudaError_t launch_one(const StageParams<T>& p, int sm_count, cudaStream_t s) {
  using G = Geo<NW>;
  const size_t smem = (size_t)G::TOTAL * sizeof(T);
  static bool configured = false;     // per instantiation; the attribute is per function and sticks
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute((const void*)stage_fused_kernel<T, LIM, NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  const int bx = (p.nx + TX - 1) / TX, by = (p.ny + G::TY - 1) / G::TY;
  // z chunk: long enough that the 4 lead-in planes are cheap, short enough that the grid fills the GPU
  int ZL = 64;
  while (ZL > 8 && (long long)bx * by * ((p.nz + ZL - 1) / ZL) < 4LL * sm_count) ZL >>= 1;
  const int bz = (p.nz + ZL - 1) / ZL;
  dim3 grid(bx, by, bz), block(NW * 32);
  stage_fused_kernel<T, LIM, NW><<<grid, block, smem, s>>>(p, ZL);
  return cudaGetLastError();
}

}  // namespace

template <class T>
cudaError_t launch_stage_fused(const StageParams<T>& p, int limiter, int sm_count, cudaStream_t s, bool* supported) {
  // packs are two cells adjacent in x: nx must be even; in-plane offsets are 32-bit; grid.y/z <= 65535
  *supported = (p.nx % 2 == 0) && ((long long)p.nx * p.ny < (1LL << 31)) && ((p.ny + 6) / 7 <= 65535);
  if (!*supported) return cudaSuccess;
  switch (limiter) {
    case 1: return launch_one<T, 1, 8>(p, sm_count, s);
    case 2: return launch_one<T, 2, 8>(p, sm_count, s);
    default: return launch_one<T, 0, 8>(p, sm_count, s);
  }
}

template cudaError_t launch_stage_fused<float>(const StageParams<float>&, int, int, cudaStream_t, bool*);
template cudaError_t launch_stage_fused<double>(const StageParams<double>&, int, int, cudaStream_t, bool*);

}  // namespace dh
