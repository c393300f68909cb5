// dh_probe.cu — dh_issue_probe: a measurement, not part of the path.  It times short instruction mixes of the kind the
// stage kernels are made of (half-rate ALU-pipe instructions: FMNMX / LOP3 / FSEL; scalar fp32 FADD / FFMA; the packed
// FADD2 / FMUL2 / FFMA2 of sm_100 in the operand forms the kernels use) on every SM, with 2 or 4 warps per scheduler and
// 8 independent dependency chains per thread, and reports SM cycles per instruction group per scheduler.
// §7b derives the issue bound of stage_fused2_kernel from this table (bench.py --issue-probe prints it;
// profiles/r02d_issue_bound.md holds the B200 numbers): a packed instruction occupies the issue port for as many cycles
// as it has distinct register-pair sources, so packing halves the instruction count but not the issue time.
//
// Every mix is a loop of `iters` x 16 groups; a group is the instruction sequence named by the mix (inline PTX, volatile,
// loop-carried through its own registers so that nothing can be hoisted).  Cycles come from clock64() of one lane per
// block (max over the blocks), not from an assumed clock.
#include <cstdio>

#include "../../include/dh.h"
#include "dh_internal.cuh"

namespace dh {
void set_error(const char* where, const char* detail);   // dh_api.cu
}

namespace dh {
namespace {

constexpr int NCH = 8;   // independent chains per thread

#define DH_P_ALU1(i) asm volatile("min.xorsign.abs.f32 %0, %0, 0f7F000000;" : "+f"(a[i]));                      /* FMNMX, 1 register source */
#define DH_P_ALU2(i) asm volatile("min.xorsign.abs.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(b[i]));                  /* FMNMX, 2 register sources */
#define DH_P_LOP(i) asm volatile("lop3.b32 %0, %0, %1, 0x80000000, 0xf8;" : "+r"(u[i]) : "r"(v[i]));            /* LOP3 */
#define DH_P_SEL(i) asm volatile("{ .reg .pred q; setp.ne.s32 q, %2, 0; selp.f32 %0, %0, %1, q; }" : "+f"(a[i]) : "f"(b[i]), "r"(pr));
#define DH_P_FADD(i) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(b[i]) : "f"(s0));                             /* scalar FADD */
#define DH_P_FFMA(i) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(b[i]) : "f"(a[i]), "f"(e[i]));            /* scalar FFMA, 3 registers */
#define DH_P_FFMAI(i) asm volatile("fma.rn.f32 %0, %0, 0f3F800347, %0;" : "+f"(b[i]));                          /* scalar FFMA, 1 register + immediate */
#define DH_P_F2_3(i) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(p[i]) : "l"(q[i]), "l"(r[i]));          /* FFMA2, 3 register pairs */
#define DH_P_F2_BC(i) asm volatile("{ .reg .b64 t; mov.b64 t, {%2, %2}; fma.rn.f32x2 %0, t, %1, %0; }" : "+l"(p[i]) : "l"(q[i]), "f"(s0));   /* FFMA2, broadcast scalar + 2 pairs */
#define DH_P_F2_IMM(i) asm volatile("{ .reg .b64 t; mov.b64 t, {0fBF000000, 0fBF000000}; fma.rn.f32x2 %0, %1, t, %0; }" : "+l"(p[i]) : "l"(q[i]));   /* FFMA2, immediate + 2 pairs */
#define DH_P_M2_2(i) asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(p[i]) : "l"(q[i]));                         /* FMUL2, 2 register pairs */
#define DH_P_A2_2(i) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[i]) : "l"(q[i]));                         /* FADD2, 2 register pairs */
#define DH_P_F2_1(i) asm volatile("fma.rn.f32x2 %0, %0, %0, %0;" : "+l"(p[i]));                                 /* FFMA2, 1 register pair */
#define DH_P_NONE(i)

#define DH_P_BODY(M_, X, Y, Z)                                                         \
  else if (MIX == M_) {                                                                \
    for (int it = 0; it < iters; ++it) {                                               \
      _Pragma("unroll") for (int rep = 0; rep < 2; ++rep)                              \
      _Pragma("unroll") for (int i = 0; i < NCH; ++i) { X(i) Y(i) Z(i) }               \
    }                                                                                  \
  }

template <int MIX>
__global__ void __launch_bounds__(512, 1) issue_probe_kernel(long long* cycles, float* sink, int iters, float s0, float s1, int pr) {
  float a[NCH], b[NCH], e[NCH];
  unsigned u[NCH], v[NCH];
  unsigned long long p[NCH], q[NCH], r[NCH];
#pragma unroll
  for (int i = 0; i < NCH; ++i) {
    a[i] = s0 + i + threadIdx.x; b[i] = s1 * 0.5f + i; e[i] = s1 - 0.25f * i * threadIdx.x; u[i] = threadIdx.x * i; v[i] = threadIdx.x + i;
    asm("mov.b64 %0, {%1, %2};" : "=l"(p[i]) : "f"(a[i]), "f"(b[i]));
    asm("mov.b64 %0, {%1, %2};" : "=l"(q[i]) : "f"(b[i]), "f"(a[i]));
    asm("mov.b64 %0, {%1, %2};" : "=l"(r[i]) : "f"(s1 - i), "f"(s0 * i));
  }
  __syncthreads();
  const long long t0 = clock64();
  if (false) {}
  DH_P_BODY(0, DH_P_ALU1, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(1, DH_P_LOP, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(2, DH_P_SEL, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(3, DH_P_FADD, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(4, DH_P_FFMA, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(5, DH_P_FFMAI, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(6, DH_P_F2_1, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(7, DH_P_M2_2, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(8, DH_P_A2_2, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(9, DH_P_F2_IMM, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(10, DH_P_F2_BC, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(11, DH_P_F2_3, DH_P_NONE, DH_P_NONE)
  DH_P_BODY(12, DH_P_ALU1, DH_P_FADD, DH_P_NONE)
  DH_P_BODY(13, DH_P_ALU1, DH_P_FFMAI, DH_P_FFMAI)
  DH_P_BODY(14, DH_P_ALU1, DH_P_FFMA, DH_P_NONE)
  DH_P_BODY(15, DH_P_ALU1, DH_P_F2_1, DH_P_NONE)
  DH_P_BODY(16, DH_P_ALU1, DH_P_M2_2, DH_P_NONE)
  DH_P_BODY(17, DH_P_ALU1, DH_P_F2_IMM, DH_P_NONE)
  DH_P_BODY(18, DH_P_ALU1, DH_P_F2_BC, DH_P_NONE)
  DH_P_BODY(19, DH_P_ALU1, DH_P_F2_3, DH_P_NONE)
  DH_P_BODY(20, DH_P_ALU2, DH_P_F2_3, DH_P_NONE)
  DH_P_BODY(21, DH_P_ALU1, DH_P_FFMA, DH_P_M2_2)
  DH_P_BODY(22, DH_P_ALU1, DH_P_FFMA, DH_P_F2_3)
  DH_P_BODY(23, DH_P_ALU1, DH_P_ALU1, DH_P_M2_2)
  const long long t1 = clock64();
  float s = 0;
#pragma unroll
  for (int i = 0; i < NCH; ++i) {
    float x, y;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(p[i]));
    s += a[i] + b[i] + e[i] + x + y + (float)u[i];
  }
  sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

struct MixInfo {
  const char* name;
  int instructions;   // per group
};
const MixInfo kMixes[DH_ISSUE_PROBE_MIXES] = {
    {"FMNMX (1 reg)", 1}, {"LOP3", 1}, {"FSEL", 1}, {"FADD (reg, const)", 1}, {"FFMA (3 regs)", 1}, {"FFMA (reg, imm)", 1},
    {"FFMA2 (1 pair)", 1}, {"FMUL2 (2 pairs)", 1}, {"FADD2 (2 pairs)", 1}, {"FFMA2 (2 pairs, imm)", 1}, {"FFMA2 (2 pairs, scalar)", 1}, {"FFMA2 (3 pairs)", 1},
    {"FMNMX + FADD (reg, const)", 2}, {"FMNMX + 2 FFMA (reg, imm)", 3}, {"FMNMX + FFMA (3 regs)", 2}, {"FMNMX + FFMA2 (1 pair)", 2}, {"FMNMX + FMUL2 (2 pairs)", 2},
    {"FMNMX + FFMA2 (2 pairs, imm)", 2}, {"FMNMX + FFMA2 (2 pairs, scalar)", 2}, {"FMNMX + FFMA2 (3 pairs)", 2}, {"FMNMX (2 regs) + FFMA2 (3 pairs)", 2},
    {"FMNMX + FFMA + FMUL2", 3}, {"FMNMX + FFMA + FFMA2 (3 pairs)", 3}, {"2 FMNMX + FMUL2", 3},
};

template <int MIX>
cudaError_t launch_probe(int threads, int blocks, long long* cyc, float* sink, int iters, cudaStream_t s) {
  issue_probe_kernel<MIX><<<blocks, threads, 0, s>>>(cyc, sink, iters, 1.0f, 1.5f, 1);
  return cudaGetLastError();
}

template <int MIX>
struct Dispatch {
  static cudaError_t go(int mix, int threads, int blocks, long long* cyc, float* sink, int iters, cudaStream_t s) {
    if (mix == MIX) return launch_probe<MIX>(threads, blocks, cyc, sink, iters, s);
    return Dispatch<MIX - 1>::go(mix, threads, blocks, cyc, sink, iters, s);
  }
};
template <>
struct Dispatch<-1> {
  static cudaError_t go(int, int, int, long long*, float*, int, cudaStream_t) { return cudaErrorInvalidValue; }
};

}  // namespace
}  // namespace dh

extern "C" {

const char* dh_issue_probe_name(int mix) {
  if (mix < 0 || mix >= DH_ISSUE_PROBE_MIXES) return nullptr;
  return dh::kMixes[mix].name;
}

int dh_issue_probe(int mix, int warps_per_scheduler, int iters, double* cycles_per_group, int* instructions_per_group) {
  using namespace dh;
  if (mix < 0 || mix >= DH_ISSUE_PROBE_MIXES || warps_per_scheduler < 1 || warps_per_scheduler > 4 || iters < 1 || !cycles_per_group) {
    set_error("dh_issue_probe", "mix in [0, DH_ISSUE_PROBE_MIXES), warps_per_scheduler in 1..4, iters >= 1, cycles_per_group non-NULL");
    return DH_ERR_ARG;
  }
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
    set_error("dh_issue_probe", "no CUDA device");
    return DH_ERR_CUDA;
  }
  const int threads = 128 * warps_per_scheduler;
  long long* cyc = nullptr;
  float* sink = nullptr;
  if (cudaMalloc(&cyc, sizeof(long long) * sms) != cudaSuccess || cudaMalloc(&sink, sizeof(float) * sms * threads) != cudaSuccess) {
    cudaFree(cyc);
    set_error("dh_issue_probe", "cudaMalloc failed");
    return DH_ERR_CUDA;
  }
  cudaError_t e = Dispatch<DH_ISSUE_PROBE_MIXES - 1>::go(mix, threads, sms, cyc, sink, 64, nullptr);   // warm-up (instruction cache, clocks)
  if (e == cudaSuccess) e = Dispatch<DH_ISSUE_PROBE_MIXES - 1>::go(mix, threads, sms, cyc, sink, iters, nullptr);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  long long worst = 0;
  if (e == cudaSuccess) {
    long long* h = new long long[sms];
    e = cudaMemcpy(h, cyc, sizeof(long long) * sms, cudaMemcpyDeviceToHost);
    for (int i = 0; i < sms; ++i) worst = h[i] > worst ? h[i] : worst;
    delete[] h;
  }
  cudaFree(cyc);
  cudaFree(sink);
  if (e != cudaSuccess) {
    set_error("dh_issue_probe", cudaGetErrorString(e));
    return DH_ERR_CUDA;
  }
  // groups per scheduler: warps_per_scheduler warps x iters x 16 groups each
  *cycles_per_group = (double)worst / ((double)warps_per_scheduler * iters * 16.0);
  if (instructions_per_group) *instructions_per_group = kMixes[mix].instructions;
  return DH_OK;
}

}  // extern "C"
