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

// S6 for one record by one WARP (only the last block of a request runs it).  Same outputs as emit_record
// (dyplan_common.cuh), which one thread walks node by node with two dependent global loads and a 64-bit division per
// node; here lane n takes node n -- option counts, the digit of the winner's canonical index, the option's annotations
// -- so the record costs two round trips to L2 instead of two per node.  C64 is still the product in node order, by
// one lane, without contraction (definition 4; matches the plain definition bit for bit).
// (ob, K, vn: node `lane`'s first option, option count and vulnerability, fetched by the caller before it reduced the
// records, so that their round trip is not in front of this one's)
__device__ __noinline__ void emit_small(const CallArgs& a, const ReqHdr* h, long long r, int l, const Best& w, int ob, unsigned long long K, float vn) {
  const int lane = threadIdx.x & 31;
  if (w.idx == kNoIdx) {   // warp-uniform
    if (lane == 0) emit_record(a, h, r, l, w);
    return;
  }
  const dyplan_batch& b = a.in;
  const dyplan_bundle& o = a.out;
  const int B = b.B, M = b.M;
  const long long rec = r * a.L + l;
  const int N = h->n_orig;
  unsigned long long stride = K;   // inclusive prefix product over the lanes, then shifted: stride of node `lane`
#pragma unroll
  for (int off = 1; off < 16; off <<= 1) {
    const unsigned long long t = __shfl_up_sync(0xffffffffu, stride, off);
    if (lane >= off) stride *= t;
  }
  stride = __shfl_up_sync(0xffffffffu, stride, 1);
  if (lane == 0) stride = 1;
  int k = 0;
  if (lane < N) k = ((w.idx | stride) >> 32) == 0 ? (int)(((uint32_t)w.idx / (uint32_t)stride) % (uint32_t)K) : (int)((w.idx / stride) % K);
  double f = 1.0;
  int be = 0, mo = 0, dm = 0;
  if (lane < 16) o.choice[rec * 16 + lane] = lane < N ? (uint8_t)k : (uint8_t)0xFF;
  if (lane < N && !((h->skip_mask >> lane) & 1)) {
    const int op = ob + k;
    f = __dsub_rn(1.0, __dmul_rn((double)vn, __dsub_rn(1.0, (double)b.acc[op])));
    be = b.backend[op]; mo = b.model[op]; dm = b.demand[op];
  }
  double c = 1.0;
  int D[DYPLAN_MAX_BACKENDS], Dm[DYPLAN_MAX_MODELS];
#pragma unroll
  for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) D[i] = 0;
#pragma unroll
  for (int i = 0; i < DYPLAN_MAX_MODELS; i++) Dm[i] = 0;
  for (int n = 0; n < N; n++) {   // node order (skipped nodes carry f = 1, demand 0)
    c = __dmul_rn(c, __shfl_sync(0xffffffffu, f, n));
    const int bn = __shfl_sync(0xffffffffu, be, n), mn = __shfl_sync(0xffffffffu, mo, n), dn = __shfl_sync(0xffffffffu, dm, n);
#pragma unroll
    for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) D[i] += (i == bn) ? dn : 0;
#pragma unroll
    for (int i = 0; i < DYPLAN_MAX_MODELS; i++) Dm[i] += (i == mn) ? dn : 0;
  }
  if (lane != 0) return;
  int dmod = 0, dbest = Dm[0];
#pragma unroll
  for (int m = 1; m < DYPLAN_MAX_MODELS; m++) if (m < M && Dm[m] > dbest) { dbest = Dm[m]; dmod = m; }   // ties -> lowest id (reading Q13)
  o.plan_idx[rec] = w.idx;
  o.corr[rec] = w.C;
  if (o.corr64) o.corr64[rec] = c;
  o.lat[rec] = w.T;
#pragma unroll
  for (int bb = 0; bb < DYPLAN_MAX_BACKENDS; bb++) if (bb < B) o.dem[rec * B + bb] = D[bb];
  o.dom_model[rec] = (uint8_t)dmod;
  o.status[rec] = DYPLAN_ST_OK;
}

// Plans [p, pe) of one request, from scratch, one after the other: NPB bounds the node count, so that the digits, the
// slots and the slacks are registers (a node loop with a run-time bound put them in local memory: 0.7 M local accesses
// per launch on configs[0]).  deps(i) only holds nodes j > i and is the same for every thread of the block, so the slack
// recurrence is a chain of predicated minima with uniform predicates.  The canonical index is only formed for a plan
// that is not already worse than the incumbent on (C, T).
template <int NPB>
__device__ __forceinline__ void small_walk(const uint32_t* __restrict__ sb, const int L, const bool caps, uint32_t p, const uint32_t pe, Best (&best)[DYPLAN_MAX_LEVELS]) {
  const ReqHdr* h = (const ReqHdr*)sb;
  const int nsp = h->nslots_pad, Np = h->n_int, slo = h->slo;
  const int* s_lat = (const int*)(sb + kHdrWords + kDem0bWords);   // [slot][L]
  const float* s_f = (const float*)(s_lat + nsp * L);
  const int* s_dem = (const int*)(s_f + nsp);
  const int* s_be = s_dem + nsp;
  int dig[NPB], rad[NPB], ob[NPB];
  uint32_t dep[NPB];
  {
    uint32_t q = p;
#pragma unroll
    for (int i = 0; i < NPB; i++) {
      rad[i] = i < Np ? (i == 0 ? h->K0 : (i == 1 ? h->K1 : h->Kp[i])) : 1;
      ob[i] = i < Np ? h->optbase[i] : 0;
      dep[i] = i < Np ? h->deps[i] : 0u;
      dig[i] = (int)(q % (uint32_t)rad[i]);
      q /= (uint32_t)rad[i];
    }
  }
  for (; p < pe; p++) {
    // definition 4 (as every scorer rounds it: the fp32 product from the last internal node down), 5 and 1
    float C = 1.0f;
    int D[DYPLAN_MAX_BACKENDS];
#pragma unroll
    for (int b = 0; b < DYPLAN_MAX_BACKENDS; b++) D[b] = 0;
    int sl[NPB];   // slot of node i's option
#pragma unroll
    for (int i = NPB - 1; i >= 0; --i) {
      sl[i] = ob[i] + dig[i];
      if (i < Np) {
        C = __fmul_rn(C, s_f[sl[i]]);
        if (caps) {
          const int be = s_be[sl[i]] & 7, dm = s_dem[sl[i]];
#pragma unroll
          for (int b = 0; b < DYPLAN_MAX_BACKENDS; b++) D[b] += (b == be) ? dm : 0;
        }
      }
    }
    bool capok = true;
    if (caps) {
#pragma unroll
      for (int b = 0; b < DYPLAN_MAX_BACKENDS; b++) capok = capok && D[b] <= h->cap[b];
    }
    if (capok) {
      unsigned long long idx = kNoIdx;   // formed on first use
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) {
        if (l < L) {
          // definitions 2-3 in slack form: u[i] = min(SLO, min_{j in deps(i)} u[j]) - d_l(i, k_i), T = SLO - min_i u[i]
          int u[NPB];
          int ms = slo;
#pragma unroll
          for (int i = NPB - 1; i >= 0; --i) {
            u[i] = slo;
            if (i < Np) {
              int m = slo;
#pragma unroll
              for (int j = i + 1; j < NPB; j++) if ((dep[i] >> j) & 1u) m = min(m, u[j]);
              const int v = m - s_lat[sl[i] * L + l];
              u[i] = v;
              ms = min(ms, v);
            }
          }
          const int T = slo - ms;
          if (ms >= 0 && (best[l].idx == kNoIdx || C > best[l].C || (C == best[l].C && T <= best[l].T))) {
            if (idx == kNoIdx) {
              idx = h->base_idx;
#pragma unroll
              for (int i = 0; i < NPB; i++) if (i < Np) idx += (unsigned long long)dig[i] * h->stride[i];
            }
            if (better(C, T, idx, best[l])) { best[l].C = C; best[l].T = T; best[l].idx = idx; }
          }
        }
      }
    }
#pragma unroll
    for (int i = 0; i < NPB; i++) {   // odometer
      if (++dig[i] < rad[i]) break;
      dig[i] = 0;
    }
  }
}

// (`a` is a __grid_constant__: the not-inlined emit_small takes it by reference, and without the qualifier every thread
// first copied the 1.2 KB argument block to its local memory -- 100 STL.128 per warp, 126 MB of local stores per launch)
__global__ void __launch_bounds__(kSmallThreads, 4) k_small(const __grid_constant__ CallArgs a) {
  __shared__ __align__(16) uint32_t sb[kMaxBlobWords];
  __shared__ Best s_red[DYPLAN_MAX_LEVELS][kSmallThreads / 32];
  __shared__ uint32_t s_last;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int split = a.small_split;
  const long long r = blockIdx.x / split;
  const int part = blockIdx.x % split;
  const int L = a.L;
  const uint32_t* gblob = a.blob + (size_t)r * blob_stride_words(L);
  // the header says how long the blob is, but reading it first would put two round trips to L2 in front of every
  // block: the first 5 x 128 words (header, dem0b and 35 slots at 3 levels) are fetched unconditionally, the rest after
  constexpr int kFirst = 5 * kSmallThreads;
#pragma unroll
  for (int i = 0; i < 5; i++) sb[tid + i * kSmallThreads] = gblob[tid + i * kSmallThreads];
  __syncthreads();
  const ReqHdr* h = (const ReqHdr*)sb;
  if (h->status != DYPLAN_ST_OK || h->klass != kClassSmall) return;   // block-uniform
  const int words = kHdrWords + kDem0bWords + h->nslots_pad * (L + 3);
  if (words > kFirst) {   // block-uniform
    for (int i = kFirst + tid; i < words; i += kSmallThreads) sb[i] = gblob[i];
    __syncthreads();
  }
  const int Np = h->n_int;

  // this thread's contiguous range of enumerated plans (internal mixed radix, node 0 fastest); P <= 2^21
  const uint32_t P = (uint32_t)(h->outer_total * (unsigned long long)(h->K0 * h->K1));
  const uint32_t nthr = (uint32_t)split * kSmallThreads;
  const uint32_t chunk = (P + nthr - 1) / nthr;
  const uint32_t gt = (uint32_t)part * kSmallThreads + tid;
  const uint32_t p = gt * chunk < P ? gt * chunk : P;
  const uint32_t pe = p + chunk < P ? p + chunk : P;
  Best best[DYPLAN_MAX_LEVELS];
#pragma unroll
  for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) { best[l].C = -1.0f; best[l].T = INT32_MAX; best[l].idx = kNoIdx; }
  // (one instantiation per bound on the node count: digits, slots and slacks stay in registers)
  const bool caps = a.in.cap != nullptr;
  if (Np <= 4) small_walk<4>(sb, L, caps, p, pe, best);
  else if (Np <= 6) small_walk<6>(sb, L, caps, p, pe, best);
  else if (Np <= 8) small_walk<8>(sb, L, caps, p, pe, best);
  else if (Np <= 12) small_walk<12>(sb, L, caps, p, pe, best);
  else small_walk<16>(sb, L, caps, p, pe, best);

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
  // ---- last block of this request (S6): warp l takes level l -- the records of all parts with ten loads in flight per
  // lane (two round trips for 592 parts), shuffles, and the same warp emits; the node constants the emission needs are
  // fetched first, so their round trip overlaps the records'.  (Measured on configs[0]: this tail was 15 us of the
  // kernel's 27 when one thread block walked the levels one after the other and the emission fetched on its own.) ----
  const int n_orig = h->n_orig;
  int e_ob = 0; unsigned long long e_K = 1; float e_v = 0.0f;
  if (wid < L && lane < n_orig) {
    e_ob = a.in.opt_off[h->n0 + lane];
    e_K = (unsigned long long)(a.in.opt_off[h->n0 + lane + 1] - e_ob);
    e_v = a.in.vuln[h->n0 + lane];
  }
  for (int l = wid; l < L; l += kSmallThreads / 32) {
    Best v; v.C = -1.0f; v.T = INT32_MAX; v.idx = kNoIdx;
    for (int j0 = lane; j0 < split; j0 += 32 * 10) {
      float4 raw[10];
#pragma unroll
      for (int q = 0; q < 10; q++) {
        const int j = j0 + 32 * q;
        raw[q] = j < split ? __ldcg((const float4*)&part_rec[(size_t)j * L + l]) : make_float4(-1.0f, __int_as_float(INT32_MAX), __uint_as_float(0xffffffffu), __uint_as_float(0xffffffffu));
      }
#pragma unroll
      for (int q = 0; q < 10; q++) {
        Best o; o.C = raw[q].x; o.T = __float_as_int(raw[q].y);
        o.idx = ((unsigned long long)__float_as_uint(raw[q].w) << 32) | (unsigned long long)__float_as_uint(raw[q].z);
        if (better(o.C, o.T, o.idx, v)) v = o;
      }
    }
    v = warp_best(v);
    emit_small(a, h, r, l, v, e_ob, e_K, e_v);
  }
  if (tid == 0) { atomicAdd(&a.st->total_plans, (unsigned long long)P); atomicAdd(&a.st->small_requests, 1u); }   // (k_plan sets the totals again when the general scorers run too)
}

cudaError_t launch_small(const CallArgs& a, cudaStream_t s) {
  if (a.in.R == 0) return cudaSuccess;
  k_small<<<(unsigned)(a.in.R * a.small_split), kSmallThreads, 0, s>>>(a);
  return cudaGetLastError();
}

}  // namespace dyplan
