// dyplan_small.cu -- K_small: the admission-time path.  One request compiled alone ("execution starts as soon as pi^(0)
// is ready") is a latency problem, not a throughput problem: the batched scorers' machinery (incumbent
// seeds, work items, a persistent grid, the cooperative exact re-walk) costs 0.15 ms on BASELINE configs[0], all of it
// fixed latency.  For calls of at most kSmallMaxR requests, every request whose enumerated space is at most 2^21
// (plan, level) evaluations is staged in the int32 layout with class kClassSmall and solved here, the same definitions
// written out per plan: `small_split` blocks per request (the call's requests share about four
// blocks per SM: a lone warp per scheduler runs at a sixth of the issue rate), each thread scores a contiguous range
// of plans from scratch in the internal node order -- C32 as the fp32 product from the last internal node down (the
// order every scorer uses, so C32 is the same pure function of the plan), the slack form of Eq.(3) and the demand sums
// in int32 -- and keeps its own arg-best per level under order 7; warp shuffles, shared memory, one record per (block,
// level), a ticket, and the last block of the request reduces and emits the bundle records.  No seeds, no screen.
#include "dyplan_common.cuh"

namespace dyplan {

// (not inlined: only the last block of a request runs it)
__device__ __noinline__ void emit_small(const CallArgs& a, const ReqHdr* h, long long r, int l, const Best& w) { emit_record(a, h, r, l, w); }

__global__ void __launch_bounds__(kSmallThreads) k_small(const CallArgs a) {
  __shared__ __align__(16) uint32_t sb[kMaxBlobWords];
  __shared__ Best s_red[DYPLAN_MAX_LEVELS][kSmallThreads / 32];
  __shared__ uint32_t s_last;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int split = a.small_split;
  const long long r = blockIdx.x / split;
  const int part = blockIdx.x % split;
  const int L = a.L;
  const uint32_t* gblob = a.blob + (size_t)r * blob_stride_words(L);
  const ReqHdr* gh = (const ReqHdr*)gblob;
  if (gh->status != DYPLAN_ST_OK || gh->klass != kClassSmall) return;   // block-uniform
  const int words = kHdrWords + kDem0bWords + gh->nslots_pad * (L + 3);
  for (int i = tid; i < words; i += kSmallThreads) sb[i] = gblob[i];
  __syncthreads();
  const ReqHdr* h = (const ReqHdr*)sb;
  const int nsp = h->nslots_pad, Np = h->n_int, slo = h->slo;
  const int* s_lat = (const int*)(sb + kHdrWords + kDem0bWords);   // [slot][L]
  const float* s_f = (const float*)(s_lat + nsp * L);
  const int* s_dem = (const int*)(s_f + nsp);
  const int* s_be = s_dem + nsp;

  // this thread's contiguous range of enumerated plans (internal mixed radix, node 0 fastest); P <= 2^21
  const uint32_t P = (uint32_t)(h->outer_total * (unsigned long long)(h->K0 * h->K1));
  const uint32_t nthr = (uint32_t)split * kSmallThreads;
  const uint32_t chunk = (P + nthr - 1) / nthr;
  const uint32_t gt = (uint32_t)part * kSmallThreads + tid;
  uint32_t p = gt * chunk < P ? gt * chunk : P;
  const uint32_t pe = p + chunk < P ? p + chunk : P;
  int dig[16], rad[16];
  {
    uint32_t q = p;
    for (int i = 0; i < Np; i++) {
      rad[i] = i == 0 ? h->K0 : (i == 1 ? h->K1 : h->Kp[i]);
      dig[i] = (int)(q % (uint32_t)rad[i]);
      q /= (uint32_t)rad[i];
    }
  }
  Best best[DYPLAN_MAX_LEVELS];
#pragma unroll
  for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) { best[l].C = -1.0f; best[l].T = INT32_MAX; best[l].idx = kNoIdx; }

  for (; p < pe; p++) {
    // definition 4 (as every scorer rounds it), 5 and 1
    float C = 1.0f;
    int D[DYPLAN_MAX_BACKENDS];
#pragma unroll
    for (int b = 0; b < DYPLAN_MAX_BACKENDS; b++) D[b] = 0;
    unsigned long long idx = h->base_idx;
    for (int i = Np - 1; i >= 0; --i) {
      const int slot = h->optbase[i] + dig[i];
      C = __fmul_rn(C, s_f[slot]);
      const int be = s_be[slot] & 7, dm = s_dem[slot];
#pragma unroll
      for (int b = 0; b < DYPLAN_MAX_BACKENDS; b++) D[b] += (b == be) ? dm : 0;
      idx += (unsigned long long)dig[i] * h->stride[i];
    }
    bool capok = true;
#pragma unroll
    for (int b = 0; b < DYPLAN_MAX_BACKENDS; b++) capok = capok && D[b] <= h->cap[b];
    if (capok) {
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) {
        if (l < L) {
          // definitions 2-3 in slack form: u[i] = min(SLO, min_{j in deps(i)} u[j]) - d_l(i, k_i), T = SLO - min_i u[i]
          int u[16];
          int ms = slo;
          for (int i = Np - 1; i >= 0; --i) {
            int m = slo;
            for (uint32_t dm = h->deps[i]; dm; dm &= dm - 1) m = min(m, u[__ffs(dm) - 1]);
            const int v = m - s_lat[(h->optbase[i] + dig[i]) * L + l];
            u[i] = v;
            ms = min(ms, v);
          }
          if (ms >= 0 && better(C, slo - ms, idx, best[l])) { best[l].C = C; best[l].T = slo - ms; best[l].idx = idx; }
        }
      }
    }
    for (int i = 0; i < Np; i++) {   // odometer
      if (++dig[i] < rad[i]) break;
      dig[i] = 0;
    }
  }

  // ---- block arg-best per level, one record per (request, part, level) ----
#pragma unroll
  for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) {
    if (l >= L) break;
    const Best v = warp_best(best[l]);
    if (lane == 0) s_red[l][wid] = v;
  }
  __syncthreads();
  Partial* part_rec = a.partial + ((size_t)r * split) * L;
  if (tid < L) {
    Best v = s_red[tid][0];
    for (int w = 1; w < kSmallThreads / 32; w++) { const Best o = s_red[tid][w]; if (better(o.C, o.T, o.idx, v)) v = o; }
    Partial q; q.C = v.C; q.T = v.T; q.idx = v.idx;
    part_rec[(size_t)part * L + tid] = q;
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();   // release in the ticket-taking thread, after the block barrier
    s_last = (atomicAdd(&a.done[r], 1u) == (uint32_t)split - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  for (int l = wid; l < L; l += kSmallThreads / 32) {
    // ---- last block of this request: a warp reduces one level's records and emits (S6) ----
    Best v; v.C = -1.0f; v.T = INT32_MAX; v.idx = kNoIdx;
    for (int j = lane; j < split; j += 32) {
      const float4 raw = __ldcg((const float4*)&part_rec[(size_t)j * L + l]);
      Best o; o.C = raw.x; o.T = __float_as_int(raw.y);
      o.idx = ((unsigned long long)__float_as_uint(raw.w) << 32) | (unsigned long long)__float_as_uint(raw.z);
      if (better(o.C, o.T, o.idx, v)) v = o;
    }
    v = warp_best(v);
    if (lane == 0) emit_small(a, h, r, l, v);
  }
  if (tid == 0) { atomicAdd(&a.st->total_plans, (unsigned long long)P); atomicAdd(&a.st->small_requests, 1u); }   // (k_plan sets the totals again when the general scorers run too)
}

cudaError_t launch_small(const CallArgs& a, cudaStream_t s) {
  if (a.in.R == 0) return cudaSuccess;
  k_small<<<(unsigned)(a.in.R * a.small_split), kSmallThreads, 0, s>>>(a);
  return cudaGetLastError();
}

}  // namespace dyplan
