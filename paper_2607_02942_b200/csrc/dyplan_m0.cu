// dyplan_m0.cu -- M0: measured issue rates of the instructions the scorers are built from (SURVEY.md section 7 step 5,
// 8(d) D.3; include/dyplan.h dyplan_measure_issue_rates).  The roofline of this path is instruction issue on the plain
// FP32/INT32 pipes, and MEASURED_PEAKS.json records only HBM and tensor peaks, so the denominator is measured here.
//
// One kernel per instruction (template on the opcode): every thread runs kChains independent dependency chains of that
// one instruction in a fully unrolled block of kBlockInst instructions, kIters times.  One block per SM, kWarpsPerSmsp
// warps per SMSP.  A warp stamps clock64() before and after its loop; the rate of an SM is
//     (warps * kIters * kBlockInst) / 4 SMSPs / (latest end - earliest start)      warp-instructions / clk / SMSP
// and the reported figure is the median over the SMs.  The loop's own counter/branch instructions (2 per kBlockInst
// payload instructions) are not counted: the figure is a slight under-estimate of the pipe's rate (< 2 %).
// The SM clock actually held is (cycles of the longest block) / (CUDA-event time of the launch).
#include "dyplan_internal.cuh"

namespace dyplan {

constexpr int kM0Chains = 8;        // independent chains per thread
constexpr int kM0BlockInst = 128;   // payload instructions per loop iteration (16 per chain)
constexpr int kM0Iters = 2048;
constexpr int kM0WarpsPerSmsp = 8;

enum M0Op { M0_FFMA = 0, M0_FADD_SAT, M0_FMUL, M0_FADD, M0_FMNMX3, M0_IADD3, M0_VIADDMNMX, M0_VIMNMX3, M0_IMAD, M0_LOP3, M0_MIX_SCREEN, M0_MIX_INT, M0_FFMA2, M0_FADD2, M0_FMUL2, M0_MIX_SCREEN2, M0_COUNT };

template <int OP>
__device__ __forceinline__ void m0_step(float (&f)[kM0Chains], int (&i)[kM0Chains], float c0, float c1, int k0, int k1) {
#pragma unroll
  for (int c = 0; c < kM0Chains; c++) {
    if (OP == M0_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(c0), "f"(c1));
    if (OP == M0_FADD_SAT) asm volatile("add.sat.f32 %0, %0, %1;" : "+f"(f[c]) : "f"(c1));
    if (OP == M0_FMUL) asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(f[c]) : "f"(c0));
    if (OP == M0_FADD) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[c]) : "f"(c1));
    if (OP == M0_FMNMX3) asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(c0), "f"(c1));
    if (OP == M0_IADD3) asm volatile("{ .reg .s32 t; add.s32 t, %0, %1; add.s32 %0, t, %2; }" : "+r"(i[c]) : "r"(k0), "r"(k1));
    if (OP == M0_VIADDMNMX) i[c] = __viaddmax_s32(i[c], k0, k1);
    if (OP == M0_VIMNMX3) i[c] = __vimax3_s32(i[c], k0, k1);
    if (OP == M0_IMAD) asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(i[c]) : "r"(k0), "r"(k1));
    if (OP == M0_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(i[c]) : "r"(k0), "r"(k1));
  }
}

// the screen's own mix: per two (plan, level) evaluations 2 FADD.SAT + 2 FFMA + 1 FMNMX3 (dyplan_fscore.cuh); the
// products feed the next step's adds, so nothing is loop-invariant
__device__ __forceinline__ void m0_mix_screen(float (&f)[kM0Chains], float (&g)[kM0Chains], float c0, float c1, float c2) {
#pragma unroll
  for (int c = 0; c < kM0Chains; c += 2) {
    float x0, x1, z0, z1;
    asm volatile("add.sat.f32 %0, %1, %2;" : "=f"(x0) : "f"(f[c]), "f"(c1));
    asm volatile("add.sat.f32 %0, %1, %2;" : "=f"(x1) : "f"(f[c + 1]), "f"(c2));
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(z0) : "f"(x0), "f"(c0), "f"(-c2));
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(z1) : "f"(x1), "f"(c0), "f"(-c1));
    asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(g[c >> 1]) : "f"(z0), "f"(z1));
    f[c] = z0; f[c + 1] = z1;
  }
}

// the int32 screen of the wide class: IADD3 + FFMA + LOP3 per evaluation (dyplan_score.cuh)
__device__ __forceinline__ void m0_mix_int(float (&f)[kM0Chains], int (&i)[kM0Chains], float c0, float c1, int k0) {
#pragma unroll
  for (int c = 0; c < kM0Chains; c++) {
    int t; float y;
    asm volatile("sub.s32 %0, %1, %2;" : "=r"(t) : "r"(i[c]), "r"(k0));
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(y) : "f"(f[c]), "f"(c0), "f"(c1));
    asm volatile("lop3.b32 %0, %0, %1, %2, 0xE0;" : "+r"(i[c]) : "r"(t), "r"(__float_as_int(y)));
    f[c] = y;
  }
}

// packed fp32 (sm_100: FFMA2 / FADD2 / FMUL2 work on an aligned register pair): kM0Chains / 2 chains of pairs
__device__ __forceinline__ unsigned long long m0_pack(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void m0_unpack(unsigned long long v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }

template <int OP>
__device__ __forceinline__ void m0_step2(unsigned long long (&p)[kM0Chains / 2], unsigned long long c0, unsigned long long c1) {
#pragma unroll
  for (int c = 0; c < kM0Chains / 2; c++) {
    if (OP == M0_FFMA2) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[c]) : "l"(c0), "l"(c1));
    if (OP == M0_FADD2) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(c1));
    if (OP == M0_FMUL2) asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(c0));
  }
}

// the screen with the product and the incumbent test of TWO evaluations in one FFMA2: per two (plan, level)
// evaluations 2 FADD.SAT + 1 FFMA2 + 1 FMNMX3
__device__ __forceinline__ void m0_mix_screen2(float (&f)[kM0Chains], float (&g)[kM0Chains], unsigned long long c00, unsigned long long cneg, float c1, float c2) {
#pragma unroll
  for (int c = 0; c < kM0Chains; c += 2) {
    float x0, x1, z0, z1;
    asm volatile("add.sat.f32 %0, %1, %2;" : "=f"(x0) : "f"(f[c]), "f"(c1));
    asm volatile("add.sat.f32 %0, %1, %2;" : "=f"(x1) : "f"(f[c + 1]), "f"(c2));
    unsigned long long z = m0_pack(x0, x1);
    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(z) : "l"(c00), "l"(cneg));
    m0_unpack(z, z0, z1);
    asm volatile("max.f32 %0, %0, %1, %2;" : "+f"(g[c >> 1]) : "f"(z0), "f"(z1));
    f[c] = z0; f[c + 1] = z1;
  }
}

template <int OP>
__global__ void __launch_bounds__(kM0WarpsPerSmsp * 4 * 32, 1) k_m0(long long* __restrict__ stamps, float* __restrict__ sink, float c0, float c1, int k0, int k1) {
  float f[kM0Chains], g[kM0Chains];
  int i[kM0Chains];
#pragma unroll
  for (int c = 0; c < kM0Chains; c++) { f[c] = 0.25f + 0.001f * (float)(threadIdx.x + c); g[c] = 0.0f; i[c] = (int)threadIdx.x + c; }
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < kM0Iters; it++) {
    if (OP == M0_MIX_SCREEN) {
      // 5 instructions per pair of chains -> 20 per call; 6 calls + 8 payload = 128
#pragma unroll
      for (int rep = 0; rep < 6; rep++) m0_mix_screen(f, g, c0, c1, c0 + c1);
#pragma unroll
      for (int c = 0; c < 8; c++) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(c0), "f"(c1));
    } else if (OP == M0_MIX_SCREEN2) {
      // 4 instructions per pair of chains -> 16 per call; 8 calls = 128
      const unsigned long long c00 = m0_pack(c0, c0), cneg = m0_pack(-(c0 + c1), -c1);
#pragma unroll
      for (int rep = 0; rep < 8; rep++) m0_mix_screen2(f, g, c00, cneg, c1, c0 + c1);
    } else if (OP == M0_FFMA2 || OP == M0_FADD2 || OP == M0_FMUL2) {
      unsigned long long p[kM0Chains / 2];
#pragma unroll
      for (int c = 0; c < kM0Chains / 2; c++) p[c] = m0_pack(f[2 * c], f[2 * c + 1]);
      const unsigned long long c00 = m0_pack(c0, c0), c11 = m0_pack(c1, c1);
#pragma unroll
      for (int rep = 0; rep < kM0BlockInst / (kM0Chains / 2); rep++) m0_step2<OP>(p, c00, c11);
#pragma unroll
      for (int c = 0; c < kM0Chains / 2; c++) m0_unpack(p[c], f[2 * c], f[2 * c + 1]);
    } else if (OP == M0_MIX_INT) {
      // 3 instructions per chain -> 24 per call; 5 calls + 8 payload = 128
#pragma unroll
      for (int rep = 0; rep < 5; rep++) m0_mix_int(f, i, c0, c1, k0);
#pragma unroll
      for (int c = 0; c < 8; c++) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(c0), "f"(c1));
    } else {
#pragma unroll
      for (int rep = 0; rep < kM0BlockInst / kM0Chains; rep++) m0_step<OP>(f, i, c0, c1, k0, k1);
    }
  }
  const long long t1 = clock64();
  float acc = 0.0f;
#pragma unroll
  for (int c = 0; c < kM0Chains; c++) acc += f[c] + g[c] + (float)i[c];
  if (acc == 1.2345e-30f) sink[0] = acc;   // keeps the chains alive; never true in practice
  if ((threadIdx.x & 31) == 0) {
    const int w = threadIdx.x >> 5;
    stamps[((size_t)blockIdx.x * (blockDim.x >> 5) + w) * 2 + 0] = t0;
    stamps[((size_t)blockIdx.x * (blockDim.x >> 5) + w) * 2 + 1] = t1;
  }
}

typedef void (*m0_kernel_t)(long long*, float*, float, float, int, int);
static const m0_kernel_t kM0Kernels[M0_COUNT] = {
    k_m0<M0_FFMA>, k_m0<M0_FADD_SAT>, k_m0<M0_FMUL>, k_m0<M0_FADD>, k_m0<M0_FMNMX3>, k_m0<M0_IADD3>,
    k_m0<M0_VIADDMNMX>, k_m0<M0_VIMNMX3>, k_m0<M0_IMAD>, k_m0<M0_LOP3>, k_m0<M0_MIX_SCREEN>, k_m0<M0_MIX_INT>,
    k_m0<M0_FFMA2>, k_m0<M0_FADD2>, k_m0<M0_FMUL2>, k_m0<M0_MIX_SCREEN2>};
static const char* const kM0Names[M0_COUNT] = {
    "FFMA", "FADD.SAT", "FMUL", "FADD", "FMNMX3", "IADD3", "VIADDMNMX", "VIMNMX3", "IMAD", "LOP3",
    "mix: 2 FADD.SAT + 2 FFMA + 1 FMNMX3 (k_fscore screen)", "mix: IADD3 + FFMA + LOP3 (k_score screen)",
    "FFMA2 (packed: 2 FMA per lane)", "FADD2 (packed)", "FMUL2 (packed)", "mix: 2 FADD.SAT + 1 FFMA2 + 1 FMNMX3 (packed screen)"};

int m0_count() { return M0_COUNT; }
const char* m0_name(int op) { return (op >= 0 && op < M0_COUNT) ? kM0Names[op] : ""; }
int m0_warps_per_block() { return kM0WarpsPerSmsp * 4; }
double m0_warp_inst_per_warp() { return (double)kM0Iters * (double)kM0BlockInst; }
cudaError_t m0_launch(int op, int grid, long long* stamps, float* sink, cudaStream_t s) {
  kM0Kernels[op]<<<grid, kM0WarpsPerSmsp * 4 * 32, 0, s>>>(stamps, sink, 0.999f, 1e-3f, 3, 5);
  return cudaGetLastError();
}

}  // namespace dyplan
