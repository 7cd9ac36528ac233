// dyplan_stage.cu -- K_stage (validate + stage per-request tables) and K_plan (work decomposition).
// SURVEY.md 8(a) S0; Alg. 1 l.1-8 "coefficient construction" is the paper's counterpart.
#include "dyplan_internal.cuh"

namespace dyplan {

__device__ __forceinline__ void write_sentinel(const dyplan_bundle& o, long long rec, int B, int status) {
  o.plan_idx[rec] = kNoIdx;
  for (int i = 0; i < 16; i++) o.choice[rec * 16 + i] = 0xFF;
  o.corr[rec] = -1.0f;
  if (o.corr64) o.corr64[rec] = -1.0;
  o.lat[rec] = INT32_MAX;
  for (int b = 0; b < B; b++) o.dem[rec * B + b] = 0;
  o.dom_model[rec] = 0xFF;
  o.status[rec] = (uint8_t)status;
}

__device__ __forceinline__ int k0_class(int k) { return k <= 2 ? 2 : k <= 4 ? 4 : k <= 6 ? 6 : k <= 8 ? 8 : k <= 12 ? 12 : 16; }

// definition 2 (reading Q4): d_l(n,k) = floor(tau * mult / 1000) in int64
__device__ __forceinline__ long long scaled(int tau, int mult) { return ((long long)tau * (long long)mult) / 1000; }

// f = 1 - v (1 - a) in fp64 without contraction (f = v * r^, r^ = 1 - q)
__device__ __forceinline__ double factor64(float v, float a) { return __dsub_rn(1.0, __dmul_rn((double)v, __dsub_rn(1.0, (double)a))); }

// index of the k-th set bit of m (k < popcount(m))
__device__ __forceinline__ int nth_set_bit(uint32_t m, int k) {
  for (int i = 0; i < k; i++) m &= m - 1;
  return __ffs(m) - 1;
}

// Exact per-node dominance pruning: option x of a node can be dropped when another
// option y of the same node is at least as good in every quantity the objective reads -- factor f (as the scorer's
// fp32 value), every level's scaled duration, and with caps the same backend and no more demand -- and the plan with y
// in place of x is STRICTLY preferred by the order the scorer applies: (C32 desc, T asc, idx asc), C32 being the fp32
// product in the scorer's fixed node order.  Rounding is monotone, so fy >= fx gives C32(y-plan) >= C32(x-plan) and
// T(y-plan) <= T(x-plan); that is strict when y < x (lower canonical index breaks the last tie).  For y > x the index
// speaks for x, so C32 itself must separate: the exact products differ by the factor fy / fx, each fp32 product of
// <= 16 factors is within 16 * 2^-24 of exact, hence fy >= fx (1 + 2^-18) (3.8e-6 > 2 * 0.96e-6) keeps
// C32(y-plan) > C32(x-plan).  (Factors a few ulps apart -- tiny v -- round to equal products; x then wins the tie-break
// of the full enumeration and must be kept.)  The relation is transitive and acyclic: every dropped option is
// dominated by a kept one, and no dropped option is in any best plan.
__device__ uint32_t dominance_keep(const dyplan_batch& b, int o0, int K, float v, const int* mult, int L, int B, bool has_caps) {
  uint32_t keep = K >= 32 ? 0xffffffffu : ((1u << K) - 1u);
  for (int x = 0; x < K; x++) {
    const int ox = o0 + x;
    const float fx = (float)factor64(v, b.acc[ox]);
    for (int y = 0; y < K; y++) {
      if (y == x) continue;
      const int oy = o0 + y;
      if (has_caps && (b.backend[oy] != b.backend[ox] || b.demand[oy] > b.demand[ox])) continue;
      const float fy = (float)factor64(v, b.acc[oy]);
      const bool separated = (double)fy >= __dmul_rn((double)fx, 1.0 + 1.0 / 262144.0) && fy > fx;
      if (!(separated || (fy >= fx && y < x))) continue;
      bool ok = true;
      for (int l = 0; l < L && ok; l++)
        ok = scaled(b.lat_us[oy], mult[l * B + b.backend[oy]]) <= scaled(b.lat_us[ox], mult[l * B + b.backend[ox]]);
      if (ok) { keep &= ~(1u << x); break; }
    }
  }
  return keep;
}

// One warp per request.
__global__ void __launch_bounds__(128) k_stage(CallArgs a) {
  const int lane = threadIdx.x & 31;
  if (a.img_src) {
    // a tiny *_host call: its inputs (a few hundred bytes) arrive as one image in pinned host memory, and every block
    // fetches the whole of it itself (one round trip over the host link; blocks write identical bytes) instead of the
    // call paying a DMA copy and its stream-order hand-over in front of this kernel
    for (uint32_t i = threadIdx.x; i < a.img_vec; i += blockDim.x) a.img_dst[i] = a.img_src[i];
    __syncthreads();
  }
  const long long r = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const dyplan_batch& b = a.in;
  if (r >= b.R) return;
  const int L = a.L, B = b.B;
  const size_t blob_stride = blob_stride_words(L);
  uint32_t* blob = a.blob + (size_t)r * blob_stride;
  ReqHdr* h = (ReqHdr*)blob;
  const int* mult = a.is_replan ? a.mult + (size_t)r * B : a.mult;

  if (lane == 0) a.done[r] = 0;
  if (lane < L) a.gthr[r * L + lane] = 0.0f;
  if (r == 0 && lane == 0) {   // (k_small adds to total_plans; k_plan, when it runs, sets every field)
    CallState* st = a.st;
    st->total_plans = 0; st->total_outer = 0; st->slow_steps = 0; st->bound_skipped = 0; st->total_items = 0; st->total_items_f = 0;
    st->next_item = 0; st->next_item_f = 0; st->fast_requests = 0; st->approx_requests = 0; st->small_requests = 0;
  }

  // ---- shape checks, in the oracle's order (load_req, validate, dispatched set, size of the free space) ----
  int st = DYPLAN_ST_OK;
  long long sum_lat = 0, sum_dem = 0;   // largest possible T over the levels / largest possible total demand
  double min_c = 1.0;                   // smallest possible C (product of the per-node minimum factors)
  const int n0 = b.node_off[r], n1 = b.node_off[r + 1];
  const int N = n1 - n0;
  int K[16], o0[16];
  unsigned long long stride[16];
#pragma unroll
  for (int n = 0; n < 16; n++) { K[n] = 1; o0[n] = 0; stride[n] = 0; }
  if (N < 0 || N > DYPLAN_MAX_NODES || n0 < 0 || n1 > b.NN) st = DYPLAN_ST_INVALID;
  if (st == DYPLAN_ST_OK) {
    unsigned long long s = 1;
#pragma unroll
    for (int n = 0; n < 16; n++) {
      if (n < N && st == DYPLAN_ST_OK) {
        o0[n] = b.opt_off[n0 + n];
        K[n] = b.opt_off[n0 + n + 1] - o0[n];
        if (K[n] < 1 || K[n] > DYPLAN_MAX_OPTS || o0[n] < 0 || o0[n] + K[n] > b.KK) { st = DYPLAN_ST_INVALID; K[n] = 1; }
        else {
          stride[n] = s;
          if (__umul64hi(s, (unsigned long long)K[n]) != 0ull || s * (unsigned long long)K[n] > (1ull << 60)) st = DYPLAN_ST_TOO_LARGE;   // s K > 2^60, without a division
          s *= (unsigned long long)K[n];
        }
      }
    }
  }
  if (st == DYPLAN_ST_OK) {
    bool bad = false;
    for (int i = lane; i < L * B; i += 32) bad |= mult[i] < 0;
    if (lane == 0) bad |= b.slo_us[r] < 0;
    if (b.cap && lane < B) bad |= b.cap[r * B + lane] < 0;
    // per-node fields: lane n
    int nodeK = 1, nodeo0 = 0;
#pragma unroll
    for (int n = 0; n < 16; n++) if (n == lane) { nodeK = K[n]; nodeo0 = o0[n]; }
    if (lane < N) {
      const uint32_t pm = b.pred_mask[n0 + lane];
      bad |= (pm >> lane) != 0;
      const float v = b.vuln[n0 + lane];
      bad |= !(v >= 0.0f && v <= 1.0f);
      for (int k = 0; k < nodeK; k++) {
        const int o = nodeo0 + k;
        bad |= b.lat_us[o] < 0 || b.demand[o] < 0;
        const float ac = b.acc[o];
        bad |= !(ac >= 0.0f && ac <= 1.0f);
        bad |= b.backend[o] >= B || b.model[o] >= b.M;
      }
    }
    bad = __any_sync(0xffffffffu, bad);
    if (!bad) {
      // reading Q19: sum_n max_k d_l and sum_n max_k demand must fit int32
      for (int l = 0; l <= L && !bad; l++) {
        long long mx = 0;
        if (lane < N)
          for (int k = 0; k < nodeK; k++) {
            const int o = nodeo0 + k;
            const long long d = (l < L) ? scaled(b.lat_us[o], mult[l * B + b.backend[o]]) : (long long)b.demand[o];
            mx = d > mx ? d : mx;
          }
#pragma unroll
        for (int off = 16; off; off >>= 1) mx += __shfl_xor_sync(0xffffffffu, mx, off);
        bad |= mx > (long long)INT32_MAX;
        if (l < L) sum_lat = mx > sum_lat ? mx : sum_lat; else sum_dem = mx;
      }
      // smallest possible C: the fp32 scorer needs every plan's C32 to be a positive normal number
      if (!bad) {
        double mn = 1.0;
        if (lane < N) {
          const float v = b.vuln[n0 + lane];
          for (int k = 0; k < nodeK; k++) { const double f = factor64(v, b.acc[nodeo0 + k]); mn = f < mn ? f : mn; }
        }
#pragma unroll
        for (int off = 16; off; off >>= 1) mn *= __shfl_xor_sync(0xffffffffu, mn, off);
        min_c = mn;
      }
    }
    if (bad) st = DYPLAN_ST_INVALID;
  }
  uint32_t fmask = 0;
  if (st == DYPLAN_ST_OK && a.is_replan) {
    fmask = a.dispatched[r];
    bool bad = (N < 32) && ((fmask >> N) != 0);
    if (!bad && lane < N && ((fmask >> lane) & 1)) {
      int nodeK = 1;
#pragma unroll
      for (int n = 0; n < 16; n++) if (n == lane) nodeK = K[n];
      bad |= a.fixed_choice[n0 + lane] >= nodeK;
      bad |= (b.pred_mask[n0 + lane] & ~fmask) != 0;   // reading Q11: predecessor-closed
    }
    bad = __any_sync(0xffffffffu, bad);
    if (bad) st = DYPLAN_ST_INVALID;
  }
  if (st != DYPLAN_ST_OK) {
    if (lane == 0) { h->status = st; h->outer_total = 0; h->nslots_pad = 0; h->K0 = 1; h->K1 = 1; }
    if (lane < L) write_sentinel(a.out, r * L + lane, B, st);
    return;
  }

  // ---- internal order ----
  const int Kfirst = N ? (((fmask >> 0) & 1) ? 1 : K[0]) : 1;
  int Klast = 1;
#pragma unroll
  for (int n = 0; n < 16; n++) if (n == N - 1) Klast = ((fmask >> n) & 1) ? 1 : K[n];
  const int orient = (N >= 1 && Klast > Kfirst) ? 1 : 0;
  const int Np = N < 3 ? 3 : N;
  const bool residual = a.is_replan && (a.flags & DYPLAN_RESIDUAL);

  // lane i < Np describes internal node i
  int e = -1;
  if (lane < N) e = orient ? N - 1 - lane : lane;
  int myK = 1, myo0 = 0; unsigned long long mystride = 0;
#pragma unroll
  for (int n = 0; n < 16; n++) if (n == e) { myK = K[n]; myo0 = o0[n]; mystride = stride[n]; }
  const bool fixed = e >= 0 && ((fmask >> e) & 1);
  const int fk = fixed ? a.fixed_choice[n0 + e] : 0;
  uint32_t deps = 0;
  if (e >= 0) {
    if (!orient) {
      for (int j = e + 1; j < N; j++) if ((b.pred_mask[n0 + j] >> e) & 1) deps |= 1u << j;
    } else {
      const uint32_t pm = b.pred_mask[n0 + e];
      for (int p = 0; p < e; p++) if ((pm >> p) & 1) deps |= 1u << (N - 1 - p);
    }
  }

  // ---- scorer class: the fp32 scorer takes a request when every slack and demand sum is an exact
  // fp32 integer, node 0's options fit its backend-grouped slot layout and the tables fit its shared-memory window ----
  const int Lp = level_class(L);
  const bool has_caps = b.cap != nullptr;
  const int nbc = !has_caps ? 0 : (B <= 2 ? 2 : (B == 3 ? 3 : (B == 4 ? 4 : 8)));
  // the fp32 scorer is exact when every slack / demand sum is an integer below 2^23; beyond that its slacks are upper
  // bounds (directed rounding) and candidates are verified with int32 tables (ReqHdr.approx)
  // small call, small request: the int32 layout, solved by k_small without seeds, items or a persistent grid
  bool small = false;
  if (a.small_mode) {
    unsigned long long pf = (e >= 0 && !fixed) ? (unsigned long long)myK : 1ull;   // <= 16^16: no overflow
#pragma unroll
    for (int off = 16; off; off >>= 1) {
      const unsigned long long o = __shfl_xor_sync(0xffffffffu, pf, off);
      pf = (pf > kSmallMaxEvals || o > kSmallMaxEvals) ? kSmallMaxEvals + 1 : pf * o;
    }
    small = pf * (unsigned long long)L <= kSmallMaxEvals;
  }
  const bool fast_pre = min_c >= 1e-30 && !small;
  const bool approx = !(sum_lat <= (1ll << 22) && (!has_caps || sum_dem <= (1ll << 22)));
  // options kept per node: all of them, or (opt-in, fast class only) the ones no other option dominates
  const uint32_t keep_full = (e >= 0 && !fixed) ? (myK >= 32 ? 0xffffffffu : ((1u << myK) - 1u)) : 1u;
  uint32_t keep = keep_full;
  bool pruned = (a.ctx_flags & DYPLAN_PRUNE_DOMINATED) && fast_pre;
  if (pruned && e >= 0 && !fixed && myK > 1) keep = dominance_keep(b, myo0, myK, b.vuln[n0 + e], mult, L, B, has_caps);
  const int e0 = __shfl_sync(0xffffffffu, e, 0), K0all = __shfl_sync(0xffffffffu, myK, 0), o00 = __shfl_sync(0xffffffffu, myo0, 0);
  const int fixed0 = __shfl_sync(0xffffffffu, (int)fixed, 0), fk0 = __shfl_sync(0xffffffffu, fk, 0);
  int Kp = 1, K0r = 1, K1r = 1, G = 0, K0p = 2, width = 0, optbase = 0, nslots = 0, nslots_pad = 0, blob_words = 0;
  bool fast = false;
  for (int attempt = 0; attempt < 2; attempt++) {
    Kp = (e < 0 || fixed) ? 1 : __popc(keep);
    K0r = __shfl_sync(0xffffffffu, Kp, 0);
    K1r = __shfl_sync(0xffffffffu, Kp, 1);
    const uint32_t keep0 = __shfl_sync(0xffffffffu, keep, 0);
    // node 0's candidate options: its kept options, or the pinned one
    G = 0;
    if (nbc && e0 >= 0) {
      int cnt[8];
#pragma unroll
      for (int i = 0; i < 8; i++) cnt[i] = 0;
      for (int k = 0; k < K0all; k++) {
        if (fixed0 ? (k != fk0) : !((keep0 >> k) & 1)) continue;
        const int be = (fixed0 && residual) ? 0 : b.backend[o00 + k];
#pragma unroll
        for (int i = 0; i < 8; i++) cnt[i] += (be == i);
      }
#pragma unroll
      for (int i = 0; i < 8; i++) G = cnt[i] > G ? cnt[i] : G;
    } else if (nbc) G = 1;
    K0p = k0_class(K0r);
    fast = fast_pre;
    if (nbc) {
      // allowed group sizes per class: nbc*G in {2,4,6,8,12,16}
      int Gp = 0;
      if (nbc == 2) Gp = G <= 4 ? (G < 1 ? 1 : G) : (G <= 6 ? 6 : (G <= 8 ? 8 : 0));
      else if (nbc == 3) Gp = G <= 2 ? 2 : (G <= 4 ? 4 : 0);
      else if (nbc == 4) Gp = G <= 2 ? (G < 1 ? 1 : G) : (G <= 4 ? 4 : 0);
      else Gp = G <= 1 ? 1 : (G <= 2 ? 2 : 0);
      if (Gp == 0) fast = false; else if (fast) { G = Gp; K0p = nbc * Gp; }
    }
    for (int lay = 0; lay < 2; lay++) {
      width = (lane == 0) ? K0p : (lane < Np ? Kp : 0);
      optbase = width;   // inclusive scan over lanes -> exclusive
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) { int t = __shfl_up_sync(0xffffffffu, optbase, off); if (lane >= off) optbase += t; }
      nslots = __shfl_sync(0xffffffffu, optbase, 31);
      optbase -= width;
      nslots_pad = (nslots + 3) & ~3;
      blob_words = kHdrWords + nslots_pad * (Lp + 5) + (nbc ? 128 : 0);
      // (approx: the int32 tables follow in global memory and are not staged in the scorer's window)
      if (!(fast && (blob_words > kFastBlobWords || (size_t)blob_words + (approx ? nslots_pad * (Lp + 1) : 0) > blob_stride))) break;
      // tables too large for the fp32 scorer's window: fall back to the wide class (lay out again, plain inner radix)
      fast = false;
      K0p = k0_class(K0r);
    }
    if (fast || !pruned) break;
    keep = keep_full;   // pruned, but the request does not fit the fp32 scorer: the int32 scorer enumerates every option
    pruned = false;
  }
  // ---- size of the space to enumerate (after pruning, when it applies) ----
  {
    unsigned long long P = 1;
    bool too_large = false;
    for (int i = 0; i < Np; i++) {
      const unsigned long long k = (unsigned long long)__shfl_sync(0xffffffffu, Kp, i);
      if (P * k > (1ull << DYPLAN_MAX_PLANS_LOG2)) too_large = true; else P *= k;   // (P <= 2^40, k <= 16: no overflow; a 64-bit division per node cost this lone warp 2 us)
    }
    if (too_large) {
      if (lane == 0) { h->status = DYPLAN_ST_TOO_LARGE; h->outer_total = 0; h->nslots_pad = 0; h->K0 = 1; h->K1 = 1; }
      if (lane < L) write_sentinel(a.out, r * L + lane, B, DYPLAN_ST_TOO_LARGE);
      return;
    }
  }
  unsigned long long outer = (lane >= 2 && lane < Np) ? (unsigned long long)Kp : 1ull;
  unsigned long long base = fixed ? (unsigned long long)fk * mystride : 0ull;
#pragma unroll
  for (int off = 16; off; off >>= 1) { outer *= __shfl_xor_sync(0xffffffffu, outer, off); base += __shfl_xor_sync(0xffffffffu, base, off); }
  const uint32_t deps0 = __shfl_sync(0xffffffffu, deps, 0), deps1 = __shfl_sync(0xffffffffu, deps, 1);

  if (lane == 0) {
    h->status = DYPLAN_ST_OK; h->n_int = Np; h->n_orig = N; h->orient = orient; h->K0 = K0r; h->K1 = K1r; h->K0p = K0p;
    h->slo = b.slo_us[r]; h->nslots_pad = nslots_pad; h->n0 = n0; h->conn01 = (deps0 >> 1) & 1;
    h->skip_mask = residual ? fmask : 0u; h->outer_total = outer; h->base_idx = base;
    for (int bb = 0; bb < 8; bb++) h->cap[bb] = (b.cap && bb < B) ? b.cap[r * B + bb] : INT32_MAX;
    h->klass = fast ? kClassFast : (small ? kClassSmall : kClassWide); h->nbc = fast ? nbc : 0; h->Lp = Lp;
    const long long slo = b.slo_us[r];
    h->slo_f = __ll2float_ru(slo < sum_lat ? slo : sum_lat);
    h->slo_c = (int32_t)(slo < sum_lat ? slo : sum_lat);
    h->approx = (fast && approx) ? 1 : 0;
    h->ioff = kHdrWords + nslots_pad * (Lp + 5) + (nbc ? 128 : 0);
    h->pad1 = 0;
    h->S01 = ((deps0 >> 1) & 1) ? 1.0f : kBigF;
    h->big12 = ((deps1 >> 2) & 1) ? 0.0f : kBigF;
    h->big02 = ((deps0 >> 2) & 1) ? 0.0f : kBigF;
    h->blob_words = fast ? blob_words : 0;
    for (int bb = 0; bb < 8; bb++) {
      long long c = (b.cap && bb < B) ? (long long)b.cap[r * B + bb] : sum_dem;
      h->capf[bb] = __ll2float_ru(c < sum_dem ? c : sum_dem);
    }
  }
  if (lane < 16) {
    h->Kp[lane] = lane < Np ? Kp : 1;
    h->deps[lane] = lane < Np ? deps : 0;
    h->optbase[lane] = lane < Np ? optbase : 0;
    h->stride[lane] = (lane < Np && !fixed) ? mystride : 0ull;
  }

  // ---- tables.  wide: dem0b [16][8], lat [slot][L] (int32), f [slot], dem [slot], be [slot]
  //              fast: nlat [slot][Lp] (fp32, negated), f [slot], dem [slot] (fp32), be [slot], idxc [slot] (u64),
  //                    dem1b [16][8] (fp32, caps only); node 0's slots are grouped by backend when caps exist ----
  int* t_dem0b = (int*)(blob + kHdrWords);
  int* t_lat = t_dem0b + kDem0bWords;
  float* t_f = (float*)(t_lat + nslots_pad * L);
  int* t_dem = (int*)(t_f + nslots_pad);
  int* t_be = t_dem + nslots_pad;
  float* q_nlat = (float*)(blob + kHdrWords);
  float* q_f = q_nlat + nslots_pad * Lp;
  float* q_dem = q_f + nslots_pad;
  int* q_be = (int*)(q_dem + nslots_pad);
  unsigned long long* q_idxc = (unsigned long long*)(q_be + nslots_pad);
  float* q_dem1b = (float*)(q_idxc + nslots_pad);
  int* q_ilat = (int*)(q_dem1b + (nbc ? 128 : 0));   // approx only: exact durations [slot][Lp] and demands [slot]
  int* q_idem = q_ilat + nslots_pad * Lp;
  if (!fast) for (int i = lane; i < kDem0bWords; i += 32) t_dem0b[i] = 0;
  else if (nbc) for (int i = lane; i < 128; i += 32) q_dem1b[i] = 0.0f;
  __syncwarp();
  for (int s0 = 0; s0 < nslots_pad; s0 += 32) {   // uniform trip count: the body shuffles
    const int s = s0 + lane;
    const bool active = s < nslots_pad;
    // which internal node owns slot s
    int node = -1, k = 0;
    for (int i = 0; i < Np; i++) {
      const int ob = __shfl_sync(0xffffffffu, optbase, i), w = __shfl_sync(0xffffffffu, width, i);
      if (s >= ob && s < ob + w) { node = i; k = s - ob; }
    }
    // the owning node's fields, straight from its lane (a shuffle with a per-lane source)
    const int src = node < 0 ? 0 : node;
    int ne = __shfl_sync(0xffffffffu, e, src), nK = __shfl_sync(0xffffffffu, myK, src), no0 = __shfl_sync(0xffffffffu, myo0, src);
    int nfix = __shfl_sync(0xffffffffu, (int)fixed, src), nfk = __shfl_sync(0xffffffffu, fk, src);
    uint32_t nkeep = __shfl_sync(0xffffffffu, keep, src);
    unsigned long long nstride = __shfl_sync(0xffffffffu, mystride, src);
    if (node < 0) { ne = -1; nK = 1; no0 = 0; nfix = 0; nfk = 0; nkeep = 1u; nstride = 0; }
    bool pad = node < 0 || (node == 0 && k >= K0r);
    int korig = 0;   // the original option index behind slot digit k (kept options only; the pinned one for a fixed node)
    if (nfix) korig = nfk;
    else if (!pad && ne >= 0) korig = nth_set_bit(nkeep, k);
    if (fast && nbc && node == 0) {
      // slot k = group g (backend g), position p: the p-th candidate option of node 0 on backend g
      const int g = k / G, pp = k % G;
      int found = -1, seen = 0;
      for (int kk = 0; kk < nK; kk++) {
        if (nfix ? (kk != nfk) : !((nkeep >> kk) & 1)) continue;
        const int be = (ne < 0 || (nfix && residual)) ? 0 : b.backend[no0 + kk];
        if (be == g) { if (seen == pp) found = kk; seen++; }
      }
      if (ne < 0) found = (g == 0 && pp == 0) ? 0 : -1;   // dummy node: one neutral option
      pad = found < 0;
      korig = found < 0 ? 0 : found;
    }
    int dl[DYPLAN_MAX_LEVELS];
#pragma unroll
    for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) dl[l] = 0;
    float f = 1.0f; int dem = 0, be = 0;
    if (pad) {
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) dl[l] = INT32_MAX;
      f = -1.0f;   // a padding option can never tie or beat an incumbent: C1 * f <= 0
    } else if (ne >= 0 && !(nfix && residual)) {
      const int o = no0 + korig;
      be = b.backend[o]; dem = b.demand[o];
      const int tau = b.lat_us[o];
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) if (l < L) dl[l] = (int)scaled(tau, mult[l * B + be]);
      f = (float)factor64(b.vuln[n0 + ne], b.acc[o]);
    }
    if (active && !fast) {
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) if (l < L) t_lat[s * L + l] = dl[l];
      t_f[s] = f; t_dem[s] = dem; t_be[s] = be;
      if (node == 0 && !pad) t_dem0b[k * 8 + be] = dem;
    }
    if (active && fast) {
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++)
        if (l < Lp) q_nlat[s * Lp + l] = pad ? -2.0f * kBigF : __int2float_ru(-dl[l < L ? l : 0]);   // padded levels repeat level 0 (their threshold never admits a plan)
      // (negated durations rounded up and demands rounded down: exact below 2^24, else the slacks formed from them
      // are upper bounds)
      q_f[s] = pad ? 0.0f : f; q_dem[s] = __int2float_rd(dem); q_be[s] = be;
      q_idxc[s] = (pad || ne < 0 || nfix) ? 0ull : (unsigned long long)korig * nstride;
      if (nbc && node == 1 && !pad) q_dem1b[k * 8 + be] = __int2float_rd(dem);
      if (approx) {
#pragma unroll
        for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) if (l < Lp) q_ilat[s * Lp + l] = dl[l < L ? l : 0];
        q_idem[s] = dem;
      }
    }
  }
}

// ---- K_seed: seed the incumbent thresholds of the fast-class requests.  One block per request: score
// a few hundred random plans the same way k_fscore does (fp32 slack DP, C32 as the product in internal node order from
// the last node down) and publish the best feasible C per level.  A threshold is only ever the C32 of a plan that
// exists and is feasible, so the enumeration still meets that plan (ties pass the screen) and the result does not
// depend on the seeds. ----
constexpr int kSeedThreads = 128, kSeedsPerThread = 2;   // random plans per thread (plus one plan of the trade-off family)
__global__ void __launch_bounds__(kSeedThreads) k_seed(CallArgs a) {
  __shared__ __align__(16) uint32_t sb[kFastBlobWords];
  const long long r = blockIdx.x;
  const int L = a.L, B = a.in.B, tid = threadIdx.x;
  const uint32_t* blob = a.blob + (size_t)r * blob_stride_words(L);
  const ReqHdr* gh = (const ReqHdr*)blob;
  if (gh->status != DYPLAN_ST_OK || gh->klass != kClassFast) return;   // block-uniform
  const int words = gh->blob_words;
  for (int i = tid; i < words; i += kSeedThreads) sb[i] = blob[i];
  __syncthreads();
  const ReqHdr* sh = (const ReqHdr*)sb;
  const int nsp = sh->nslots_pad, Lp = sh->Lp, Np = sh->n_int, K0p = sh->K0p, nbc = sh->nbc;
  const float* p_nlat = (const float*)(sb + kHdrWords);
  const float* p_f = p_nlat + nsp * Lp;
  const float* p_dem = p_f + nsp;
  const int* p_be = (const int*)(p_dem + nsp);
  // feasibility is decided on integers in both sub-classes (exact: the fp32 tables hold integers below 2^23 and
  // convert exactly; approx: the int32 tables that follow them), so a threshold is always the C32 of a feasible plan
  const bool approx = sh->approx != 0;
  const int* p_ilat = (const int*)(blob + sh->ioff);   // (global memory: not part of blob_words)
  const int* p_idem = p_ilat + nsp * Lp;
  const int slo_c = sh->slo_c;
  int su[16][DYPLAN_MAX_LEVELS];
  // Seeds: kSeedsPerThread random plans per thread, then one plan of a one-parameter family that follows the trade-off
  // the method is about -- per node the option with the largest factor among those whose duration (at one level, the
  // thread's) is at most theta times the node's longest, theta = 1/32 .. 1 over the threads.  Random plans give a
  // threshold near the top 0.2 % of the space; a call of one or two mid-size requests then spent its time in slow-path
  // re-walks while every warp climbed from there on its own (configs[1], one request: 5931 re-walks, 0.20 ms).
  const int fam_theta = (tid & 31) + 1, fam_level = (tid >> 5) % (L > 0 ? L : 1);
  for (int sidx = 0; sidx <= kSeedsPerThread; sidx++) {
    const bool family = sidx == kSeedsPerThread;
    uint32_t x = (uint32_t)r * 0x9E3779B9u + (uint32_t)(sidx * kSeedThreads + tid) * 0x85EBCA6Bu + 0x27D4EB2Fu;
    float C = 1.0f;
    int D[8], ms[DYPLAN_MAX_LEVELS];
#pragma unroll
    for (int i = 0; i < 8; i++) D[i] = 0;
#pragma unroll
    for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) ms[l] = slo_c;
    for (int i = Np - 1; i >= 0; --i) {
      x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;   // integer hash, one draw per node
      const int kp = i == 0 ? K0p : sh->Kp[i];
      int slot = sh->optbase[i] + (int)((x >> 8) % (uint32_t)kp);
      if (family) {
        const int ob = sh->optbase[i];
        long long dmax = 0;
        for (int k = 0; k < kp; k++) {
          if (!(p_f[ob + k] > 0.0f)) continue;   // padding slot
          const long long d = approx ? (long long)p_ilat[(ob + k) * Lp + fam_level] : (long long)(-p_nlat[(ob + k) * Lp + fam_level]);
          dmax = d > dmax ? d : dmax;
        }
        const long long lim = dmax * fam_theta / 32;
        float bf = -1.0f; long long bd = 0;
        for (int k = 0; k < kp; k++) {
          const float f = p_f[ob + k];
          if (!(f > 0.0f)) continue;
          const long long d = approx ? (long long)p_ilat[(ob + k) * Lp + fam_level] : (long long)(-p_nlat[(ob + k) * Lp + fam_level]);
          if (d <= lim ? (bf < 0.0f || bd > lim || f > bf || (f == bf && d < bd)) : (bf < 0.0f || (bd > lim && d < bd))) { bf = f; bd = d; slot = ob + k; }
        }
      }
      C *= p_f[slot];
      const int be = p_be[slot] & 7;
      const int dm = approx ? p_idem[slot] : (int)p_dem[slot];
#pragma unroll
      for (int bb = 0; bb < 8; bb++) D[bb] += (bb == be) ? dm : 0;
      const uint32_t dm0 = sh->deps[i];
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++) {
        if (l < L) {
          int m = slo_c;
          for (uint32_t dmk = dm0; dmk; dmk &= dmk - 1) m = min(m, su[__ffs(dmk) - 1][l]);
          const int d = approx ? p_ilat[slot * Lp + l] : (int)(-p_nlat[slot * Lp + l]);   // (padding slot: 2^41 saturates, C = 0 anyway)
          const int v = m - d;
          su[i][l] = v;
          ms[l] = min(ms[l], v);
        }
      }
    }
    bool capok = C > 0.0f;   // a padding slot of node 0 has f = 0
    if (nbc) {
#pragma unroll
      for (int bb = 0; bb < 8; bb++) capok &= (bb >= B) || D[bb] <= sh->cap[bb];
    }
    if (capok) {
#pragma unroll
      for (int l = 0; l < DYPLAN_MAX_LEVELS; l++)
        if (l < L && ms[l] >= 0) atomicMax((int*)&a.gthr[r * L + l], __float_as_int(C));
    }
  }
}

// Single block: totals, work items per request and scorer class, exclusive scans.
// Wide class: an item is a range of outer indices handled by one block of k_score.  Fast class: an item is a range
// of outer indices handled by one warp of k_fscore.  Partial records of fast items follow those of the wide items.
__device__ __forceinline__ uint32_t block_exclusive_scan_1024(uint32_t* s_cnt, int tid, uint32_t cnt) {
  s_cnt[tid] = cnt;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {   // Hillis-Steele over 1024 entries
    uint32_t v = tid >= off ? s_cnt[tid - off] : 0;
    __syncthreads();
    s_cnt[tid] += v;
    __syncthreads();
  }
  return s_cnt[tid] - cnt;
}

__global__ void __launch_bounds__(1024) k_plan(CallArgs a) {
  __shared__ unsigned long long s_sum[1024];
  __shared__ unsigned long long s_sumf[1024];
  __shared__ unsigned long long s_plans[1024];
  __shared__ uint32_t s_cnt[1024];
  __shared__ uint32_t s_nf[1024];
  const int tid = threadIdx.x;
  const long long R = a.in.R;
  const size_t blob_stride = blob_stride_words(a.L);
  if (a.small_mode) {
    // a small call (R <= kSmallMaxR <= 32) whose requests k_small has all taken: nothing to plan.  One warp settles it
    // (the scans and reductions below cost 10 us of fixed latency, a tenth of an admission-time compile)
    __shared__ int s_other;
    if (tid == 0) s_other = 0;
    __syncthreads();
    unsigned long long pl = 0;
    uint32_t is_small = 0;
    if (tid < R) {
      const ReqHdr* h = (const ReqHdr*)(a.blob + (size_t)tid * blob_stride);
      if (h->status == DYPLAN_ST_OK) {
        if (h->klass == kClassSmall) { is_small = 1; pl = h->outer_total * (unsigned long long)(h->K0 * h->K1); }
        else s_other = 1;
      }
    }
    __syncthreads();
    if (!s_other) {   // block-uniform
      if (tid < 32) {
#pragma unroll
        for (int off = 16; off; off >>= 1) { pl += __shfl_xor_sync(0xffffffffu, pl, off); is_small += __shfl_xor_sync(0xffffffffu, is_small, off); }
      }
      if (tid <= R) { a.item_off[tid] = 0; a.item_off_f[tid] = 0; }
      if (tid == 0) {
        CallState* st = a.st;
        st->total_outer = 0; st->total_plans = pl; st->per_item_outer = kBlock; st->per_item_outer_f = 32;
        st->slow_steps = 0; st->bound_skipped = 0;
        st->total_items = 0; st->next_item = 0; st->total_items_f = 0; st->next_item_f = 0;
        st->fast_requests = 0; st->small_call_f = 1u; st->tail_start_f = 0xffffffffu; st->approx_requests = 0; st->small_requests = is_small; st->pad0 = 0;
        st->perm_nA = 0; st->perm_sA = 1; st->perm_sB = 1; st->perm_sW = 1;
      }
      return;
    }
  }
  const long long chunk = (R + 1023) / 1024;
  const long long r0 = tid * chunk, r1 = r0 + chunk < R ? r0 + chunk : R;
  unsigned long long so = 0, sf = 0, sp = 0, mxf = 0;
  uint32_t nf = 0, na = 0, ns = 0;
  __shared__ uint32_t s_na[1024];
  __shared__ uint32_t s_ns;
  __shared__ unsigned long long s_mxf;
  if (tid == 0) { s_mxf = 0; s_ns = 0; }
  __syncthreads();
  for (long long r = r0; r < r1; r++) {
    const ReqHdr* h = (const ReqHdr*)(a.blob + (size_t)r * blob_stride);
    if (h->status == DYPLAN_ST_OK) {
      if (h->klass == kClassFast) { sf += h->outer_total; nf++; na += h->approx ? 1u : 0u; mxf = h->outer_total > mxf ? h->outer_total : mxf; }
      else if (h->klass == kClassWide) so += h->outer_total;
      else ns++;
      sp += h->outer_total * (unsigned long long)(h->K0 * h->K1);
    }
  }
  s_sum[tid] = so; s_sumf[tid] = sf; s_plans[tid] = sp; s_nf[tid] = nf; s_na[tid] = na;
  if (mxf) atomicMax(&s_mxf, mxf);
  if (ns) atomicAdd(&s_ns, ns);
  __syncthreads();
  for (int off = 512; off; off >>= 1) {
    if (tid < off) { s_sum[tid] += s_sum[tid + off]; s_sumf[tid] += s_sumf[tid + off]; s_plans[tid] += s_plans[tid + off]; s_nf[tid] += s_nf[tid + off]; s_na[tid] += s_na[tid + off]; }
    __syncthreads();
  }
  const unsigned long long total_w = s_sum[0], total_f = s_sumf[0], total_plans = s_plans[0];
  const uint32_t n_fast = s_nf[0];
  __syncthreads();
  // wide: outer indices per item, a multiple of the block size; ~16K items when there is enough work
  const unsigned long long budget = a.max_items > (unsigned long long)(2 * R + 2) ? (a.max_items - (unsigned long long)(2 * R + 2)) / 2 : 1;
  unsigned long long pio = (total_w + 16383) / 16384;
  unsigned long long need = (total_w + budget - 1) / budget;
  if (need > pio) pio = need;
  pio = ((pio + kBlock - 1) / kBlock) * kBlock;
  if (pio < (unsigned long long)kBlock) pio = kBlock;
  // fast: outer indices per item, a multiple of the warp size; target_items_f items when there is enough work
  // requests of very different sizes (replan queries with 4 to 7 free nodes) balance better with more, smaller items
  const bool uneven = n_fast > 0 && s_mxf > 2 * (total_f / n_fast);
  const unsigned long long tgt0 = a.target_items_f ? a.target_items_f : 1;
  const unsigned long long tgt = uneven ? tgt0 + tgt0 / 2 : tgt0;
  unsigned long long pif = (total_f + tgt - 1) / tgt;
  need = (total_f + budget - 1) / budget;
  if (need > pif) pif = need;
  // small calls: an item should carry at least 8 outer indices per lane (its fixed cost is a few thousand instructions)
  // unless that would leave resident warps without work
  const unsigned long long warps = a.fast_warps ? a.fast_warps : 1;
  unsigned long long floor_f = (total_f + warps - 1) / warps;
  floor_f = floor_f > 256 ? 256 : floor_f;
  if (floor_f > pif) pif = floor_f;
  pif = ((pif + 31) / 32) * 32;
  if (pif < 32) pif = 32;
  const bool small_f = total_f / warps < 1024;   // not enough outer indices for one lane-aligned item per resident warp
  // A short tail: items are handed out in request order, so the last sixteenth of the requests is cut into 4x smaller
  // items and the warps finish within one small item of each other (measured per-warp exit times on configs[1]: with
  // equal items the warps idled 5.6 % of the launch at its end; last 1/4, 1/8, 1/16, 1/32 of the requests cut: 2.635 /
  // 2.589 / 2.566 / 2.563 ms; a second level of 16x smaller items lost more to the per-item prologue than it gained).
  // The exact item count decides whether the cut fits the records' buffer.
  int tail_mode = (!small_f && R >= 2 && pif >= 4 * 256) ? 1 : 0;
  uint32_t tail_start, runw, runf, total_items_w, total_items_f;
  for (;;) {
    tail_start = tail_mode >= 1 ? (uint32_t)(R - (R / 16 > 0 ? R / 16 : 1)) : 0xffffffffu;
    uint32_t cw = 0, cf = 0;
    for (long long r = r0; r < r1; r++) {
      const ReqHdr* h = (const ReqHdr*)(a.blob + (size_t)r * blob_stride);
      if (h->status != DYPLAN_ST_OK || h->klass == kClassSmall) continue;
      if (h->klass == kClassFast) { const unsigned long long q = fast_item_outer(fast_pif_of(pif, tail_start, r), h->Kp[2], small_f); cf += (uint32_t)((h->outer_total + q - 1) / q); }
      else cw += (uint32_t)((h->outer_total + pio - 1) / pio);
    }
    runw = block_exclusive_scan_1024(s_cnt, tid, cw);
    total_items_w = s_cnt[1023];
    __syncthreads();
    runf = block_exclusive_scan_1024(s_cnt, tid, cf);
    total_items_f = s_cnt[1023];
    __syncthreads();
    if (tail_mode == 0 || (unsigned long long)total_items_w + total_items_f <= (unsigned long long)a.max_items) break;   // block-uniform
    tail_mode--;
  }
  __shared__ uint32_t s_nA;
  if (tid == 0) s_nA = total_items_f;   // (no tail: every item is a regular one)
  __syncthreads();
  for (long long r = r0; r < r1; r++) {
    const ReqHdr* h = (const ReqHdr*)(a.blob + (size_t)r * blob_stride);
    a.item_off[r] = runw;
    a.item_off_f[r] = runf;
    if ((unsigned long long)r == tail_start) s_nA = runf;
    if (h->status != DYPLAN_ST_OK || h->klass == kClassSmall) continue;
    if (h->klass == kClassFast) { const unsigned long long q = fast_item_outer(fast_pif_of(pif, tail_start, r), h->Kp[2], small_f); runf += (uint32_t)((h->outer_total + q - 1) / q); }
    else runw += (uint32_t)((h->outer_total + pio - 1) / pio);
  }
  __syncthreads();
  if (tid == 1023) {
    a.item_off[R] = total_items_w;
    a.item_off_f[R] = total_items_f;
    CallState* st = a.st;
    // Hand-out order of the fast items (CallState.perm_*).  Handed out request by request, all items of a request would
    // start within microseconds of each other, each with nothing better than k_seed's threshold, and each would climb
    // to the optimum on its own through the slow path (measured: about 27 us per item on configs[1], a tenth of the
    // launch).  Strided, a request's items are spread over the whole launch and start from what the earlier ones published.
    {
      const uint32_t nA = s_nA, nB = total_items_f - s_nA;
      const uint32_t reqs = n_fast ? n_fast : 1u;
      auto stride_for = [](uint32_t n, uint32_t per_request) -> uint32_t {
        if (n <= 2) return 1u;
        uint32_t s = per_request + 1u;
        if (s >= n) s = 1u;
        for (;; s++) {
          if (s >= n) s = 1u;
          uint32_t x = n, y = s;
          while (y) { const uint32_t t = x % y; x = y; y = t; }
          if (x == 1u) return s;
        }
      };
      st->perm_nA = nA;
      st->perm_sA = stride_for(nA, (nA + reqs - 1) / reqs);
      st->perm_sB = stride_for(nB, (uint32_t)((4ull * nB + reqs - 1) / reqs));   // (a sixteenth of the requests, 4x the items each: roughly)
      st->perm_sW = stride_for(total_items_w, (uint32_t)((total_items_w + (unsigned long long)R - 1) / (unsigned long long)R));
    }
    st->total_outer = total_w + total_f; st->total_plans = total_plans; st->per_item_outer = pio; st->per_item_outer_f = pif;
    st->slow_steps = 0; st->bound_skipped = 0;
    st->total_items = total_items_w; st->next_item = 0; st->total_items_f = total_items_f; st->next_item_f = 0;
    st->fast_requests = n_fast; st->small_call_f = small_f ? 1u : 0u; st->tail_start_f = tail_start; st->approx_requests = s_na[0]; st->small_requests = s_ns; st->pad0 = 0;
  }
}

cudaError_t launch_stage(const CallArgs& a, cudaStream_t s) {
  const int wpb = 4;
  const unsigned grid = (unsigned)((a.in.R + wpb - 1) / wpb);
  if (grid == 0) return cudaSuccess;
  k_stage<<<grid, wpb * 32, 0, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_seed(const CallArgs& a, cudaStream_t s) {
  if (a.in.R == 0) return cudaSuccess;
  k_seed<<<(unsigned)a.in.R, kSeedThreads, 0, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_plan(const CallArgs& a, cudaStream_t s) {
  k_plan<<<1, 1024, 0, s>>>(a);
  return cudaGetLastError();
}

}  // namespace dyplan
