// dyplan_linear.cu -- the paper's own objective over the same plan space (include/dyplan.h
// dyplan_compile_linear): J_L = sum_n w(n,k_n) - lambda_l T - lambda_ld L D_tau, Eq.(4)/(5) PAPER.md:197-205.
//
//   k_lstage  one thread per request: validation, reach weights rho(n), w = rho q - lambda_f v (1-q)
//             - lambda_c c per option, durations as exact fp32 integers
//   k_lscore  every plan, one warp per work item (a range of outer indices of one request).  Each lane keeps its own
//             incumbent per level -- best J32 and, among the plans attaining it, min (T << 40 | idx) -- in registers; the
//             unrolled inner block only tests J >= incumbent and a group that has a hit is walked again to update.  The
//             item's record per level = max J over the lanes, min key among the lanes attaining it (shuffles).
//   k_lemit   one warp per (request, level): reduce the request's item records (J desc, key asc), decode the winner,
//             annotate, re-evaluate J in fp64
// J32 is a pure function of the plan: W is summed from the last node down, then one FFMA per term.
#include "dyplan_common.cuh"

namespace dyplan {

// order-preserving int encoding of a float (for atomicMax on the best J published per (request, level))
__device__ __forceinline__ int enc_f32(float f) { int i = __float_as_int(f); return i ^ ((i >> 31) & 0x7fffffff); }
__device__ __forceinline__ float dec_f32(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }

__global__ void __launch_bounds__(128) k_lstage(LinArgs a) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const dyplan_batch& b = a.in;
  if (r >= b.R) return;
  const int L = a.L;
  uint32_t* blob = a.blob + (size_t)r * kLinBlobWords;
  LinHdr* h = (LinHdr*)blob;
  float2* t_wd = (float2*)(blob + kLinHdrWords);   // (w, d) per slot
  for (int l = 0; l < L; l++) a.gJ[r * L + l] = enc_f32(-INFINITY);

  int st = DYPLAN_ST_OK;
  const int n0 = b.node_off[r], n1 = b.node_off[r + 1], N = n1 - n0;
  if (N < 0 || N > DYPLAN_MAX_NODES || n0 < 0 || n1 > b.NN) st = DYPLAN_ST_INVALID;
  unsigned long long P = 1, dsum = 0;
  if (st == DYPLAN_ST_OK) {
    for (int n = 0; n < N && st == DYPLAN_ST_OK; n++) {
      const int ob = b.opt_off[n0 + n], K = b.opt_off[n0 + n + 1] - ob;
      if (K < 1 || K > DYPLAN_MAX_OPTS || ob < 0 || ob + K > b.KK) { st = DYPLAN_ST_INVALID; break; }
      const uint32_t pm = b.pred_mask[n0 + n];
      const float v = b.vuln[n0 + n];
      if ((pm >> n) != 0 || !(v >= 0.0f && v <= 1.0f)) { st = DYPLAN_ST_INVALID; break; }
      int mx = 0;
      for (int k = 0; k < K; k++) {
        const int o = ob + k;
        const float q = b.acc[o], c = a.cost[o];
        if (b.lat_us[o] < 0 || !(q >= 0.0f && q <= 1.0f) || !(c >= 0.0f) || isinf(c) || b.demand[o] < 0 ||
            b.backend[o] >= b.B || b.model[o] >= b.M) { st = DYPLAN_ST_INVALID; break; }
        mx = b.lat_us[o] > mx ? b.lat_us[o] : mx;
      }
      dsum += (unsigned long long)mx;
      if (P > ((1ull << DYPLAN_MAX_PLANS_LOG2) / (unsigned long long)K)) { if (st == DYPLAN_ST_OK) st = DYPLAN_ST_TOO_LARGE; }
      else P *= (unsigned long long)K;
    }
    if (st == DYPLAN_ST_OK && dsum > (1ull << 22)) st = DYPLAN_ST_TOO_LARGE;
  }
  h->status = st; h->n_orig = N; h->n_int = N < 3 ? 3 : N; h->jmag = 0.0f;
  if (st != DYPLAN_ST_OK) {
    h->outer_total = 0;
    for (int l = 0; l < L; l++) {
      const long long rec = r * L + l;
      const dyplan_bundle& o = a.out;
      o.plan_idx[rec] = kNoIdx;
      for (int i = 0; i < 16; i++) o.choice[rec * 16 + i] = 0xFF;
      o.corr[rec] = -1.0f;
      if (o.corr64) o.corr64[rec] = -1.0;
      o.lat[rec] = INT32_MAX;
      for (int bb = 0; bb < b.B; bb++) o.dem[rec * b.B + bb] = 0;
      o.dom_model[rec] = 0xFF;
      o.status[rec] = (uint8_t)st;
      if (a.extra.dtau) a.extra.dtau[rec] = 0;
      if (a.extra.quality) a.extra.quality[rec] = -1.0;
    }
    return;
  }
  // reach sets: R(n) = {n} u R(successors), successors have larger indices
  uint32_t reach[16], succ[16];
  for (int n = 0; n < 16; n++) { reach[n] = 0; succ[n] = 0; }
  for (int s = 0; s < N; s++) {
    const uint32_t pm = b.pred_mask[n0 + s];
    for (int n = 0; n < s; n++) if ((pm >> n) & 1) succ[n] |= 1u << s;
  }
  for (int n = N - 1; n >= 0; n--) {
    uint32_t m = 1u << n;
    for (int s = n + 1; s < N; s++) if ((succ[n] >> s) & 1) m |= reach[s];
    reach[n] = m;
  }
  unsigned long long stride = 1, outer = 1;
  int slot = 0;
  const int Np = N < 3 ? 3 : N;
  float mag_w = 0.0f, mag_d = 0.0f;   // sum over the nodes of max_k |w| and of max_k d
  for (int n = 0; n < 16; n++) {
    if (n < N) {
      const int ob = b.opt_off[n0 + n], K = b.opt_off[n0 + n + 1] - ob;
      const double rho = N > 1 ? 1.0 + (double)a.p.beta * (double)a.p.effort * (double)(__popc(reach[n]) - 1) / (double)(N - 1) : 1.0;
      const double v = (double)b.vuln[n0 + n];
      h->K[n] = K; h->succ[n] = succ[n]; h->optbase[n] = slot; h->stride[n] = stride;
      for (int k = 0; k < K; k++) {
        const double q = (double)b.acc[ob + k];
        t_wd[slot + k] = make_float2((float)(rho * q - (double)a.p.lambda_f * v * (1.0 - q) - (double)a.p.lambda_c * (double)a.cost[ob + k]),
                                     (float)b.lat_us[ob + k]);
      }
      float mw = 0.0f, md = 0.0f;
      for (int k = 0; k < K; k++) { mw = fmaxf(mw, fabsf(t_wd[slot + k].x)); md = fmaxf(md, t_wd[slot + k].y); }
      mag_w += mw; mag_d += md;
      slot += K;
      stride *= (unsigned long long)K;
      if (n >= 3) outer *= (unsigned long long)K;
    } else {
      h->K[n] = 1; h->succ[n] = 0; h->optbase[n] = slot; h->stride[n] = 0;
      if (n < Np) { t_wd[slot] = make_float2(0.0f, 0.0f); slot += 1; }   // dummy node: one neutral option
    }
  }
  h->outer_total = outer;
  {
    float lv = 0.0f;
    for (int l = 0; l < L; l++) lv = fmaxf(lv, a.levels[l]);
    h->jmag = mag_w + (a.p.lambda_l + a.p.lambda_ld * lv) * mag_d;
  }
  atomicAdd(a.plans, P);
}

// One warp per work item (request r, chunk c): a range of outer indices (digits of the nodes >= 3) of the request, split
// over the lanes.  Per outer index: digits by div/mod, slack DP of the nodes >= 3 from the last node down
// (u[i] = min(0, min_succ u[j]) - d: T = -min u); then loops over the options of nodes 2, 1, 0 with one fused step each.
// One work item (request r, chunk c) for one lane of the warp; LT = padded level count, K0P = node 0's radix class.
template <int LT, int K0P>
__device__ __noinline__ void litem(const uint32_t* __restrict__ sb, const LinArgs& a, long long r, uint32_t c, const float* __restrict__ clp,
                                   float lam_l) {
  const int lane = threadIdx.x & 31;
  const int L = a.L;
  const LinHdr* h = (const LinHdr*)sb;
  const int K0 = h->K[0];
  float cl[LT];
#pragma unroll
  for (int l = 0; l < LT; l++) cl[l] = clp[l];
  const float2* t_wd = (const float2*)(sb + kLinHdrWords);   // (w, d) per slot
  const unsigned long long outer = h->outer_total;            // prod_{i>=3} K_i
  const unsigned long long per = (((outer + a.chunks - 1) / a.chunks + 31) / 32) * 32;   // a whole number of outer indices per lane
  const unsigned long long cb = min((unsigned long long)c * per, outer), ce = min(cb + per, outer);
  const unsigned long long lper = (ce - cb + 31) / 32;
  const unsigned long long ob = min(cb + lane * lper, ce), oe = min(ob + lper, ce);
  const int Np = h->n_int, K1 = h->K[1], K2 = h->K[2];
  const uint32_t succ0 = h->succ[0], succ1 = h->succ[1], succ2 = h->succ[2];
  const bool c01 = (succ0 >> 1) & 1, c02 = (succ0 >> 2) & 1, c12 = (succ1 >> 2) & 1;
  const unsigned long long st0 = h->stride[0], st1 = h->stride[1], st2 = h->stride[2];
  const int ob1 = h->optbase[1], ob2 = h->optbase[2];

  float w0[K0P], d0[K0P];         // node 0's tables in registers (padding options: w = -1e30, never an incumbent)
#pragma unroll
  for (int k = 0; k < K0P; k++) { const float2 wd = t_wd[k < K0 ? k : 0]; w0[k] = k < K0 ? wd.x : -1e30f; d0[k] = k < K0 ? wd.y : 0.0f; }
  // Tabled screen (when the table fits the register file): J - best = [cl D1 + W1 - best] + [cl d0 + w0] + lambda_l m,
  // the second bracket a constant per (option of node 0, level), the first one per (group, level).  Per evaluation that
  // leaves one FFMA and half an FMNMX3; the first bracket is added to the per-level maxima once per group.  The sum is
  // associated differently from J32 (the pure function of the plan the re-walk computes), so the screen passes
  // everything within eps of the incumbent: both chains are at most 5 roundings of partial sums no larger than jmag
  // (2^-24 each, under 2^-20 jmag together); eps = 2^-19 jmag.  The re-walk alone decides what replaces an incumbent.
  constexpr bool kTab = K0P * LT <= 32;
  float E[kTab ? K0P : 1][LT];
  if (kTab) {
#pragma unroll
    for (int k = 0; k < K0P; k++)
#pragma unroll
      for (int l = 0; l < LT; l++) E[k][l] = fmaf(cl[l], d0[k], w0[k]);
  }
  const float neg_eps = -(h->jmag * (1.0f / 524288.0f));
  float best[LT];                 // the lane's incumbent J per level and, among the plans attaining it, min (T << 40 | idx)
  unsigned long long kmin[LT];
#pragma unroll
  // the incumbent starts from the best J any finished item of this request has published: a J some plan attains, so
  // plans below it can never win and plans that tie it still pass the test (the key decides); kmin stays ~0 until
  // one of THIS lane's plans ties or beats it
  for (int l = 0; l < LT; l++) { best[l] = l < L ? dec_f32(__ldcg(&a.gJ[r * L + l])) : INFINITY; kmin[l] = ~0ull; }

  // outer nodes (>= 3): odometer over their digits; a step recomputes the slack DP, the weight / duration prefix sums and
  // the canonical index from the highest digit that changed down to node 3 (one node on average), instead of decoding
  // the outer index by div / mod and redoing every node
  float u[16], Wa[17], Da[17], Ra[17];
  unsigned long long Ia[17];
  int dig[16];
  Wa[Np] = 0.0f; Da[Np] = 0.0f; Ra[Np] = 0.0f; Ia[Np] = 0ull;
  {
    unsigned long long t = ob < oe ? ob : 0ull;
    for (int i = 3; i < Np; i++) { const unsigned long long k = (unsigned long long)h->K[i]; dig[i] = (int)(t % k); t /= k; }
  }
  int top = Np - 1;
  for (unsigned long long step = 0; step < lper; step++) {   // the same trip count on every lane: the loop shuffles
    // share the climb: every lane's incumbent rises to the best J any lane of the warp has reached (a lane whose
    // incumbent is raised by another lane's plan no longer holds a plan attaining it: its key is cleared)
#pragma unroll
    for (int l = 0; l < LT; l++) {
      float v = best[l];
#pragma unroll
      for (int off = 16; off; off >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, off));
      if (v > best[l]) { best[l] = v; kmin[l] = ~0ull; }
    }
    const unsigned long long o = ob + step;
    if (o >= oe) continue;
    for (int i = top; i >= 3; --i) {
      const float2 wd = t_wd[h->optbase[i] + dig[i]];
      float m = 0.0f;
      for (uint32_t dm = h->succ[i]; dm; dm &= dm - 1) m = fminf(m, u[__ffs(dm) - 1]);
      u[i] = m - wd.y;
      Ra[i] = fminf(Ra[i + 1], u[i]);
      Wa[i] = Wa[i + 1] + wd.x;
      Da[i] = Da[i + 1] + wd.y;
      Ia[i] = Ia[i + 1] + (unsigned long long)dig[i] * h->stride[i];
    }
    const float Wp = Wa[3], Dp = Da[3], Rm = Ra[3];
    const unsigned long long idxo = Ia[3];
    {   // advance the odometer for the next step
      int i = 3;
      for (; i < Np; i++) {
        if (++dig[i] < h->K[i]) break;
        dig[i] = 0;
      }
      top = i < Np ? i : Np - 1;
    }
    float u2in = 0.0f, u1in3 = 0.0f, a0in3 = 0.0f;
    for (uint32_t dm = succ2; dm; dm &= dm - 1) u2in = fminf(u2in, u[__ffs(dm) - 1]);
    for (uint32_t dm = succ1 & ~7u; dm; dm &= dm - 1) u1in3 = fminf(u1in3, u[__ffs(dm) - 1]);
    for (uint32_t dm = succ0 & ~7u; dm; dm &= dm - 1) a0in3 = fminf(a0in3, u[__ffs(dm) - 1]);
    for (int k2 = 0; k2 < K2; k2++) {
      const float2 wd2 = t_wd[ob2 + k2];
      const float u2 = u2in - wd2.y;
      const float R2 = fminf(Rm, u2);
      const float W2 = Wp + wd2.x, D2 = Dp + wd2.y;
      const float u1in = c12 ? fminf(u1in3, u2) : u1in3;
      const float a0in = c02 ? fminf(a0in3, u2) : a0in3;
      const unsigned long long idx2 = idxo + (unsigned long long)k2 * st2;
      for (int k1 = 0; k1 < K1; k1++) {
        const float2 wd1 = t_wd[ob1 + k1];
        const float u1 = u1in - wd1.y;
        const float R1 = fminf(R2, u1);
        const float W1 = W2 + wd1.x, D1 = D2 + wd1.y;
        const float ap = c01 ? fminf(a0in, u1) : a0in;
        const unsigned long long idx1 = idx2 + (unsigned long long)k1 * st1;
        // screen: h > = 0 iff some (plan, level) of the group ties or beats the lane's incumbent (J - best has an exact sign)
        float h = -1.0f;
        if (kTab) {
          float hm[LT];
#pragma unroll
          for (int l = 0; l < LT; l++) hm[l] = -INFINITY;
#pragma unroll
          for (int k0 = 0; k0 + 1 < K0P; k0 += 2) {
            const float ma = fminf(R1, ap - d0[k0]), mb = fminf(R1, ap - d0[k0 + 1]);   // least slack = -T
#pragma unroll
            for (int l = 0; l < LT; l++) hm[l] = fmaxf(hm[l], fmaxf(fmaf(lam_l, ma, E[k0][l]), fmaf(lam_l, mb, E[k0 + 1][l])));
          }
          float hh = -INFINITY;
#pragma unroll
          for (int l = 0; l < LT; l++) hh = fmaxf(hh, hm[l] + (fmaf(cl[l], D1, W1) - best[l]));
          h = hh >= neg_eps ? 0.0f : -1.0f;
        } else
#pragma unroll
        for (int k0 = 0; k0 < K0P; k0++) {
          const float m = fminf(R1, ap - d0[k0]);        // least slack = -T
          const float D0 = D1 + d0[k0];
          const float Jb = fmaf(lam_l, m, W1 + w0[k0]);  // W - lambda_l T
          float dj[LT];
#pragma unroll
          for (int l = 0; l < LT; l++) dj[l] = fmaf(cl[l], D0, Jb) - best[l];   // J - incumbent
#pragma unroll
          for (int l = 0; l + 1 < LT; l += 2) h = fmaxf(h, fmaxf(dj[l], dj[l + 1]));
          if (LT & 1) h = fmaxf(h, dj[LT - 1]);
        }
        if (__builtin_expect(h >= 0.0f, 0)) {
          // rare once the incumbents have risen: walk the group again and update
#pragma unroll 1
          for (int k0 = 0; k0 < K0; k0++) {
            const float2 wd0 = t_wd[k0];
            const float m = fminf(R1, ap - wd0.y);
            const float D0 = D1 + wd0.y;
            const float Jb = fmaf(lam_l, m, W1 + wd0.x);
            const unsigned long long key = ((unsigned long long)(-m) << 40) | (idx1 + (unsigned long long)k0 * st0);
#pragma unroll
            for (int l = 0; l < LT; l++) {
              const float J = fmaf(cl[l], D0, Jb);
              if (J > best[l]) { best[l] = J; kmin[l] = key; }
              else if (J == best[l] && key < kmin[l]) kmin[l] = key;
            }
          }
        }
      }
    }
  }
#pragma unroll
  for (int l = 0; l < LT; l++) {
    if (l < L) {
      // the item's record: max J over the lanes, then min key among the lanes that attain it
      float v = best[l];
#pragma unroll
      for (int off = 16; off; off >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, off));
      unsigned long long kk = best[l] == v ? kmin[l] : ~0ull;
#pragma unroll
      for (int off = 16; off; off >>= 1) { const unsigned long long o2 = __shfl_xor_sync(0xffffffffu, kk, off); kk = o2 < kk ? o2 : kk; }
      if (lane == 0) {
        LinRec rc; rc.J = v; rc.pad = 0; rc.key = kk; a.rec[((size_t)r * a.chunks + c) * L + l] = rc;
        // publish: later items of this request start from a J that one of its plans attains (ties still pass the
        // dj >= 0 test and the key decides, so the result does not depend on what is published when)
        if (kk != ~0ull) atomicMax(&a.gJ[r * L + l], enc_f32(v));
      }
    }
  }
}

template <int LT>   // LT: level count padded to 1,2,3,4,6,8 (padded levels repeat a zero weight and are dropped)
__global__ void __launch_bounds__(128, (LT <= 4 ? 4 : 3)) k_lscore(const __grid_constant__ LinArgs a) {
  __shared__ __align__(16) uint32_t s_blob[4][kLinBlobWords];
  __shared__ float s_cl[8];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t* sb = s_blob[wid];
  const int L = a.L;
  const uint32_t total = (uint32_t)a.in.R * a.chunks;
  if (threadIdx.x < 8) s_cl[threadIdx.x] = (int)threadIdx.x < L ? -(a.p.lambda_ld * a.levels[threadIdx.x]) : 0.0f;
  __syncthreads();
  const float lam_l = a.p.lambda_l;
  long long cur_req = -1;
  for (;;) {
    uint32_t item = 0;
    if (lane == 0) item = atomicAdd(&a.counter[0], 1u);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= total) break;
    // items are handed out chunk by chunk across the requests, not request by request: a request's items are then
    // spread over the whole launch and start from the J its earlier items published instead of all climbing at once
    const long long r = item % (uint32_t)a.in.R;
    const uint32_t c = item / (uint32_t)a.in.R;
    if (r != cur_req) {
      const uint32_t* blob = a.blob + (size_t)r * kLinBlobWords;
      __syncwarp();
      for (int i = lane; i < kLinBlobWords; i += 32) sb[i] = __ldg(&blob[i]);
      __syncwarp();
      cur_req = r;
    }
    const LinHdr* h = (const LinHdr*)sb;
    if (h->status != DYPLAN_ST_OK) continue;
    const int k0 = h->K[0];
    if (k0 <= 2) litem<LT, 2>(sb, a, r, c, s_cl, lam_l);
    else if (k0 <= 4) litem<LT, 4>(sb, a, r, c, s_cl, lam_l);
    else if (k0 <= 6) litem<LT, 6>(sb, a, r, c, s_cl, lam_l);
    else if (k0 <= 8) litem<LT, 8>(sb, a, r, c, s_cl, lam_l);
    else if (k0 <= 12) litem<LT, 12>(sb, a, r, c, s_cl, lam_l);
    else litem<LT, 16>(sb, a, r, c, s_cl, lam_l);
  }
}

// One warp per (request, level); lane 0 does the rest: decode the winner, annotate, re-evaluate J in fp64 (definition order of the oracle:
// W summed in node order, then - lambda_l T - lambda_ld L D_tau; no contraction).
__global__ void __launch_bounds__(128) k_lemit(LinArgs a) {
  // one WARP per record: a request with few peers is cut into thousands of items (a.chunks = 4736 for 6 requests), and
  // one thread walking them serially took 0.5 ms; the lanes stride over the item records and reduce by shuffle
  const long long rec = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  const dyplan_batch& b = a.in;
  const int L = a.L, B = b.B, M = b.M;
  if (rec >= (long long)b.R * L) return;   // warp-uniform
  const long long r = rec / L;
  const int l = (int)(rec % L);
  const LinHdr* h = (const LinHdr*)(a.blob + (size_t)r * kLinBlobWords);
  if (h->status != DYPLAN_ST_OK) return;   // sentinels were written by k_lstage
  const dyplan_bundle& o = a.out;
  float bestJ = -INFINITY;
  unsigned long long key = ~0ull;
  for (uint32_t c = lane; c < a.chunks; c += 32) {
    const LinRec rc = a.rec[((size_t)r * a.chunks + c) * L + l];
    if (rc.key == ~0ull) continue;                         // an item whose range was empty
    if (rc.J > bestJ || (rc.J == bestJ && rc.key < key)) { bestJ = rc.J; key = rc.key; }
  }
#pragma unroll
  for (int off = 16; off; off >>= 1) {
    const float oJ = __shfl_xor_sync(0xffffffffu, bestJ, off);
    const unsigned long long ok = __shfl_xor_sync(0xffffffffu, key, off);
    if (ok != ~0ull && (key == ~0ull || oJ > bestJ || (oJ == bestJ && ok < key))) { bestJ = oJ; key = ok; }
  }
  if (lane != 0) return;
  unsigned long long idx = key & ((1ull << 40) - 1);
  const int n0 = b.node_off[r], N = h->n_orig;
  uint32_t reach[16], succ[16];
  for (int n = 0; n < 16; n++) succ[n] = 0;
  for (int s = 0; s < N; s++) { const uint32_t pm = b.pred_mask[n0 + s]; for (int n = 0; n < s; n++) if ((pm >> n) & 1) succ[n] |= 1u << s; }
  for (int n = N - 1; n >= 0; n--) { uint32_t m = 1u << n; for (int s = n + 1; s < N; s++) if ((succ[n] >> s) & 1) m |= reach[s]; reach[n] = m; }
  int D[DYPLAN_MAX_BACKENDS], Dm[DYPLAN_MAX_MODELS];
  for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) D[i] = 0;
  for (int i = 0; i < DYPLAN_MAX_MODELS; i++) Dm[i] = 0;
  long long fin[16], T = 0, Dt = 0;
  double W = 0.0, qual = 1.0;
  o.plan_idx[rec] = idx;
  for (int n = 0; n < 16; n++) {
    if (n >= N) { o.choice[rec * 16 + n] = 0xFF; continue; }
    const int ob = b.opt_off[n0 + n];
    const unsigned long long K = (unsigned long long)(b.opt_off[n0 + n + 1] - ob);
    const int k = (int)(idx % K);
    idx /= K;
    o.choice[rec * 16 + n] = (uint8_t)k;
    const int op = ob + k;
    const double rho = N > 1 ? __dadd_rn(1.0, __ddiv_rn(__dmul_rn(__dmul_rn((double)a.p.beta, (double)a.p.effort), (double)(__popc(reach[n]) - 1)), (double)(N - 1))) : 1.0;
    const double q = (double)b.acc[op], v = (double)b.vuln[n0 + n];
    const double term = __dsub_rn(__dsub_rn(__dmul_rn(rho, q), __dmul_rn(__dmul_rn((double)a.p.lambda_f, v), __dsub_rn(1.0, q))),
                                  __dmul_rn((double)a.p.lambda_c, (double)a.cost[op]));
    W = __dadd_rn(W, term);
    qual = __dmul_rn(qual, __dsub_rn(1.0, __dmul_rn(v, __dsub_rn(1.0, q))));
    long long start = 0;
    const uint32_t pm = b.pred_mask[n0 + n];
    for (int uu = 0; uu < n; uu++) if ((pm >> uu) & 1) start = fin[uu] > start ? fin[uu] : start;
    fin[n] = start + b.lat_us[op];
    T = fin[n] > T ? fin[n] : T;
    Dt += b.lat_us[op];
    D[b.backend[op]] += b.demand[op];
    Dm[b.model[op]] += b.demand[op];
  }
  int dmod = 0;
  for (int m = 1; m < M; m++) if (Dm[m] > Dm[dmod]) dmod = m;
  const double J = __dsub_rn(__dsub_rn(W, __dmul_rn((double)a.p.lambda_l, (double)T)),
                             __dmul_rn(__dmul_rn((double)a.p.lambda_ld, (double)a.levels[l]), (double)Dt));
  o.corr[rec] = bestJ;
  if (o.corr64) o.corr64[rec] = J;
  o.lat[rec] = (int)T;
  for (int bb = 0; bb < B; bb++) o.dem[rec * B + bb] = D[bb];
  o.dom_model[rec] = (uint8_t)dmod;
  o.status[rec] = DYPLAN_ST_OK;
  if (a.extra.dtau) a.extra.dtau[rec] = (int)Dt;
  if (a.extra.quality) a.extra.quality[rec] = qual;
}

cudaError_t launch_linear(const LinArgs& a, int grid, cudaStream_t s) {
  if (a.in.R == 0) return cudaSuccess;
  k_lstage<<<(unsigned)((a.in.R + 127) / 128), 128, 0, s>>>(a);
  switch (level_class(a.L)) {
#define DYPLAN_LCASE(LT_) case LT_: k_lscore<LT_><<<grid, 128, 0, s>>>(a); break;
    DYPLAN_LCASE(1) DYPLAN_LCASE(2) DYPLAN_LCASE(3) DYPLAN_LCASE(4) DYPLAN_LCASE(6)
    default: k_lscore<8><<<grid, 128, 0, s>>>(a); break;
#undef DYPLAN_LCASE
  }
  const long long nrec = (long long)a.in.R * a.L;
  k_lemit<<<(unsigned)((nrec + 3) / 4), 128, 0, s>>>(a);   // one warp per record
  return cudaGetLastError();
}

}  // namespace dyplan
