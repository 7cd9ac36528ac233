// dyplan_common.cuh -- pieces shared by the two scoring kernels (k_score: int32 slack DP, k_fscore: fp32 slack DP):
// the arg-best record and its order (definition 7), warp reduction, 1-D TMA + mbarrier helpers, bundle emission (S6).
#pragma once
#include "dyplan_internal.cuh"

namespace dyplan {

struct __align__(16) Best {
  float C;
  int32_t T;
  unsigned long long idx;
};

__device__ __forceinline__ bool better(float C, int T, unsigned long long idx, const Best& b) {
  if (idx == kNoIdx) return false;
  if (b.idx == kNoIdx) return true;
  if (C != b.C) return C > b.C;
  if (T != b.T) return T < b.T;
  return idx < b.idx;
}

__device__ __forceinline__ Best warp_best(Best v) {
#pragma unroll
  for (int off = 16; off; off >>= 1) {
    Best o;
    o.C = __shfl_xor_sync(0xffffffffu, v.C, off);
    o.T = __shfl_xor_sync(0xffffffffu, v.T, off);
    o.idx = __shfl_xor_sync(0xffffffffu, v.idx, off);
    if (better(o.C, o.T, o.idx, v)) v = o;
  }
  return v;
}

// ---- TMA (1-D bulk copy) + mbarrier helpers -------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, unsigned long long* bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// ---- winner -> bundle record (S6), one thread per (request, level) ---------------------------------------------
static __device__ __forceinline__ void emit_record(const CallArgs& a, const ReqHdr* h, long long r, int l, const Best& w) {
  const dyplan_batch& b = a.in;
  const dyplan_bundle& o = a.out;
  const int B = b.B, M = b.M;
  const long long rec = r * a.L + l;
  if (w.idx == kNoIdx) {
    o.plan_idx[rec] = kNoIdx;
    for (int i = 0; i < 16; i++) o.choice[rec * 16 + i] = 0xFF;
    o.corr[rec] = -1.0f;
    if (o.corr64) o.corr64[rec] = -1.0;
    o.lat[rec] = INT32_MAX;
    for (int bb = 0; bb < B; bb++) o.dem[rec * B + bb] = 0;
    o.dom_model[rec] = 0xFF;
    o.status[rec] = DYPLAN_ST_INFEASIBLE;
    return;
  }
  const int n0 = h->n0, N = h->n_orig;
  unsigned long long idx = w.idx;
  int D[DYPLAN_MAX_BACKENDS], Dm[DYPLAN_MAX_MODELS];
  for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) D[i] = 0;
  for (int i = 0; i < DYPLAN_MAX_MODELS; i++) Dm[i] = 0;
  double c = 1.0;
  for (int n = 0; n < 16; n++) {
    if (n >= N) { o.choice[rec * 16 + n] = 0xFF; continue; }
    const int ob = b.opt_off[n0 + n];
    const unsigned long long K = (unsigned long long)(b.opt_off[n0 + n + 1] - ob);
    const int k = (int)(idx % K);
    idx /= K;
    o.choice[rec * 16 + n] = (uint8_t)k;
    if ((h->skip_mask >> n) & 1) continue;
    const int op = ob + k;
    // definition 4 in fp64, node order, no contraction (matches the plain definition bit for bit)
    c = __dmul_rn(c, __dsub_rn(1.0, __dmul_rn((double)b.vuln[n0 + n], __dsub_rn(1.0, (double)b.acc[op]))));
    D[b.backend[op]] += b.demand[op];
    Dm[b.model[op]] += b.demand[op];
  }
  int dmod = 0;
  for (int m = 1; m < M; m++) if (Dm[m] > Dm[dmod]) dmod = m;   // ties -> lowest id (reading Q13)
  o.plan_idx[rec] = w.idx;
  o.corr[rec] = w.C;
  if (o.corr64) o.corr64[rec] = c;
  o.lat[rec] = w.T;
  for (int bb = 0; bb < B; bb++) o.dem[rec * B + bb] = D[bb];
  o.dom_model[rec] = (uint8_t)dmod;
  o.status[rec] = DYPLAN_ST_OK;
}

}  // namespace dyplan
