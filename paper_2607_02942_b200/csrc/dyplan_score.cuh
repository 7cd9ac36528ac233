// dyplan_score.cuh -- K_score: enumerate + score + arg-best, one template per (L, NB).
// Included by dyplan_score_l<L>.cu with DYPLAN_SCORE_L defined.  DESIGN.md 7.2 explains the kernel (the int32 scorer of the wide class).
//
// Per work item (a range of outer indices of one request) every thread walks its outer digits in odometer
// order, keeps the slack DP of the outer nodes in local arrays, runs the middle digit (internal node 1) as a
// loop and the inner digit (internal node 0) fully unrolled with its tables in registers:
//
//   per (plan, level):   t = a'_l - d0[k0][l]            slack of the only plan-dependent path (Eq.(3) in slack form)
//                        y = C(plan) - bestC_l           sign says "not worse than the incumbent"
//                        acc &= t | bits(y)              sign(acc) stays set while no candidate showed up
//   per plan:            C = C1 * f0[k0]  (+ cap slack folded into the sign of C when caps are present)
//
// A prefix whose acc came out non-negative is re-walked by the exact slow path, which applies the full order
// (C desc, T asc, canonical index asc) and updates the thread's incumbent.
#pragma once
#include "dyplan_common.cuh"

namespace dyplan {

// ---- the per-thread walk ---------------------------------------------------------------------------------------
// Loop nest of one thread over its range of outer indices (digits of internal nodes >= 2, odometer order):
//   heavy step  (a digit >= 3 changed)  generic slack DP of nodes top..3 over local-memory arrays, then the
//                                       "node-2 context": everything node 2 / 1 / 0 need from nodes >= 3
//   light step  (digit 2)               u2, running minimum, inputs of the middle loop, C2, D2; thresholds re-read
//   middle loop (digit 1)               one fused add-min per level gives a'_l, the slack bound of node 0
//   inner block (digit 0, unrolled)     the 3-instruction screen per (plan, level); tables in registers
//   slow path   (a lane saw a candidate) exact re-walk of that K0-wide group, order 7, incumbent update
// Thresholds are shared by the block: s_thr[l] = bits of the best C found so far (any thread, plus what other
// blocks published in gthr when the item started), s_thrm[l] = bits of its float predecessor.  The screen tests
// the exact sign of C1*f0 - pred(thr) with one FFMA: fl(C1*f0) >= thr implies C1*f0 > pred(thr), so no plan that
// ties or beats the incumbent in fp32 is ever screened out.
template <int L, int K0P, int NB, bool CONN>
__device__ __noinline__ void score_range(const uint32_t* __restrict__ sb, unsigned long long o_begin, unsigned long long o_count,
                                         volatile int* s_thr, volatile int* s_thrm, Best* s_best, int* g_thr,
                                         unsigned* __restrict__ slow_io) {
  constexpr int NBX = NB ? NB : 1;
  unsigned slow_steps = 0;
  const ReqHdr* h = (const ReqHdr*)sb;
  const int nsp = h->nslots_pad;
  const int* s_dem0b = (const int*)(sb + kHdrWords);
  const int* s_lat = s_dem0b + kDem0bWords;      // [slot][L]
  const float* s_f = (const float*)(s_lat + nsp * L);
  const int* s_dem = (const int*)(s_f + nsp);
  const int* s_be = s_dem + nsp;
  const int Np = h->n_int, K0 = h->K0, K1 = h->K1, K2 = h->Kp[2], slo = h->slo;
  const int ob2 = h->optbase[2];
  const uint32_t deps0 = h->deps[0], deps1 = h->deps[1], deps2 = h->deps[2];
  const bool d0has2 = (deps0 >> 2) & 1, d1has2 = (deps1 >> 2) & 1;

  // inner tables in registers
  int d0[K0P][L];
  float f0[K0P];
  int dem0b[K0P][NBX];
#pragma unroll
  for (int k = 0; k < K0P; k++) {
#pragma unroll
    for (int l = 0; l < L; l++) d0[k][l] = s_lat[k * L + l];
    f0[k] = s_f[k];
#pragma unroll
    for (int b = 0; b < NBX; b++) dem0b[k][b] = NB ? s_dem0b[k * 8 + b] : 0;
  }
  int cap[NBX];
#pragma unroll
  for (int b = 0; b < NBX; b++) cap[b] = h->cap[b];

  // state of the nodes >= 3 (dynamic indexing -> local memory; touched once per K2*K1*K0 plans)
  int u[16][L];
  int Rm[17][L];
  float Cp[17];
  int Dp[17][NBX];
  unsigned char dig[16];
#pragma unroll
  for (int l = 0; l < L; l++) Rm[Np][l] = slo;
  Cp[Np] = 1.0f;
#pragma unroll
  for (int b = 0; b < NBX; b++) Dp[Np][b] = 0;
  {
    unsigned long long o = o_begin;
    for (int i = 2; i < Np; i++) {
      const unsigned long long kp = (unsigned long long)h->Kp[i];
      dig[i] = (unsigned char)(o % kp);
      o /= kp;
    }
  }
  int k2 = dig[2];
  int top = Np - 1;   // recompute nodes top..3
  // node-2 context
  int X2[L], Rm3[L], U1r[L], A0r[L], D3[NBX];
  float C3;
  for (;;) {
    // ---- heavy step ----
    for (int i = top; i >= 3; --i) {
      const int slot = h->optbase[i] + dig[i];
      int m[L];
#pragma unroll
      for (int l = 0; l < L; l++) m[l] = slo;
      for (uint32_t dm = h->deps[i]; dm; dm &= dm - 1) {
        const int j = __ffs(dm) - 1;
#pragma unroll
        for (int l = 0; l < L; l++) m[l] = min(m[l], u[j][l]);
      }
#pragma unroll
      for (int l = 0; l < L; l++) {
        const int v = m[l] - s_lat[slot * L + l];
        u[i][l] = v;
        Rm[i][l] = min(Rm[i + 1][l], v);
      }
      Cp[i] = Cp[i + 1] * s_f[slot];
      if (NB) {
        const int be = s_be[slot], dm = s_dem[slot];
#pragma unroll
        for (int b = 0; b < NBX; b++) Dp[i][b] = Dp[i + 1][b] + (be == b ? dm : 0);
      }
    }
#pragma unroll
    for (int l = 0; l < L; l++) { X2[l] = slo; U1r[l] = slo; A0r[l] = slo; Rm3[l] = Rm[3][l]; }
    for (uint32_t dm = deps2; dm; dm &= dm - 1) {
      const int j = __ffs(dm) - 1;
#pragma unroll
      for (int l = 0; l < L; l++) X2[l] = min(X2[l], u[j][l]);
    }
    for (uint32_t dm = deps1 & ~7u; dm; dm &= dm - 1) {
      const int j = __ffs(dm) - 1;
#pragma unroll
      for (int l = 0; l < L; l++) U1r[l] = min(U1r[l], u[j][l]);
    }
    for (uint32_t dm = deps0 & ~7u; dm; dm &= dm - 1) {
      const int j = __ffs(dm) - 1;
#pragma unroll
      for (int l = 0; l < L; l++) A0r[l] = min(A0r[l], u[j][l]);
    }
    C3 = Cp[3];
#pragma unroll
    for (int b = 0; b < NBX; b++) D3[b] = Dp[3][b];

    for (;;) {
      // ---- light step: node 2 takes option k2 ----
      const int slot2 = ob2 + k2;
      int R2[L], U1[L], A0q[L];
      float thrmf[L];
#pragma unroll
      for (int l = 0; l < L; l++) {
        const int u2 = X2[l] - s_lat[slot2 * L + l];
        R2[l] = min(Rm3[l], u2);
        U1[l] = d1has2 ? min(U1r[l], u2) : U1r[l];
        const int a0 = d0has2 ? min(A0r[l], u2) : A0r[l];
        A0q[l] = R2[l] < 0 ? R2[l] : a0;          // a node >= 2 already misses the SLO: every bound below goes negative
        thrmf[l] = __int_as_float(s_thrm[l]);
      }
      const float C2 = C3 * s_f[slot2];
      int D2[NBX];
      if (NB) {
        const int be2 = s_be[slot2], dm2 = s_dem[slot2];
#pragma unroll
        for (int b = 0; b < NBX; b++) D2[b] = D3[b] + (be2 == b ? dm2 : 0);
      }

      for (int k1 = 0; k1 < K1; k1++) {
        const int slot1 = K0P + k1;
        const float C1 = C2 * s_f[slot1];
        int slackD[NBX];
        int bad = 0;
        if (NB) {
          const int be1 = s_be[slot1], dm1 = s_dem[slot1];
#pragma unroll
          for (int b = 0; b < NBX; b++) { slackD[b] = cap[b] - D2[b] - (be1 == b ? dm1 : 0); bad |= slackD[b]; }
        }
        const float C1s = NB ? __int_as_float(__float_as_int(C1) | (bad & 0x80000000)) : C1;
        int ap[L];
#pragma unroll
        for (int l = 0; l < L; l++) {
          const int lat1 = s_lat[slot1 * L + l];
          if (CONN) ap[l] = min(U1[l] - lat1, A0q[l]);                    // one VIADDMNMX
          else { const int u1 = U1[l] - lat1; ap[l] = u1 < 0 ? u1 : A0q[l]; }
        }
        // ---- screen: K0P x L evaluations ----
        int acc0 = -1, acc1 = -1;
#pragma unroll
        for (int k0 = 0; k0 < K0P; k0++) {
          float Ck = C1s;
          if (NB) {
            int w = slackD[0] - dem0b[k0][0];
#pragma unroll
            for (int b = 1; b < NBX; b++) w = min(w, slackD[b] - dem0b[k0][b]);
            Ck = __int_as_float(__float_as_int(C1s) | (w & 0x80000000));
          }
#pragma unroll
          for (int l = 0; l < L; l++) {
            const int t = ap[l] - d0[k0][l];
            const float y = __fmaf_rn(Ck, f0[k0], -thrmf[l]);
            if ((k0 + l) & 1) acc1 &= t | __float_as_int(y);
            else acc0 &= t | __float_as_int(y);
          }
        }
        if (__builtin_expect((acc0 & acc1) >= 0, 0)) {
          // ---- slow path: exact order on this group ----
          slow_steps++;
          unsigned long long idx1 = h->base_idx + (unsigned long long)k1 * h->stride[1] + (unsigned long long)k2 * h->stride[2];
          for (int i = 3; i < Np; i++) idx1 += (unsigned long long)dig[i] * h->stride[i];
          const unsigned long long stride0 = h->stride[0];
          if (bad >= 0) {
            for (int k0 = 0; k0 < K0; k0++) {
              const float C = __fmul_rn(C1, s_f[k0]);
              if (NB) {
                int w = 0;
#pragma unroll
                for (int b = 0; b < NBX; b++) w |= slackD[b] - s_dem0b[k0 * 8 + b];
                if (w < 0) continue;
              }
              const unsigned long long idx = idx1 + (unsigned long long)k0 * stride0;
#pragma unroll
              for (int l = 0; l < L; l++) {
                const int t = ap[l] - s_lat[k0 * L + l];
                const int tb = s_thr[l];
                if (t < 0 || C < __int_as_float(tb)) continue;
                const int um = min(R2[l], U1[l] - s_lat[slot1 * L + l]);
                const int T = slo - min(t, um);
                Best* bp = &s_best[l * kBlock];
                const Best cur = *bp;
                if (better(C, T, idx, cur)) {
                  Best nb; nb.C = C; nb.T = T; nb.idx = idx;
                  *bp = nb;
                  const int cb = __float_as_int(C);
                  if (cb > tb) {
                    atomicMax((int*)&s_thr[l], cb);
                    atomicMax((int*)&s_thrm[l], cb > 0 ? cb - 1 : (int)0x80000001);
                    atomicMax(&g_thr[l], cb);
                  }
                }
              }
            }
          }
#pragma unroll
          for (int l = 0; l < L; l++) thrmf[l] = __int_as_float(s_thrm[l]);
        }
      }
      // ---- advance ----
      if (--o_count == 0) goto done;
      if (++k2 < K2) continue;
      k2 = 0;
      break;
    }
    {
      int i = 3;
      for (;;) {
        const int d = dig[i] + 1;
        if (d < h->Kp[i]) { dig[i] = (unsigned char)d; break; }
        dig[i] = 0;
        i++;
      }
      top = i;
    }
  }
done:
  *slow_io += slow_steps;
}

template <int L, int K0P, int NB>
__device__ __forceinline__ void score_dispatch(bool conn, const uint32_t* sb, unsigned long long b, unsigned long long n, volatile int* s_thr,
                                               volatile int* s_thrm, Best* s_best, int* g_thr, unsigned* slow) {
  if (conn) score_range<L, K0P, NB, true>(sb, b, n, s_thr, s_thrm, s_best, g_thr, slow);
  else score_range<L, K0P, NB, false>(sb, b, n, s_thr, s_thrm, s_best, g_thr, slow);
}

template <int L, int NB>
__global__ void __launch_bounds__(kBlock, kMinBlocks) k_score(const CallArgs a) {
  __shared__ __align__(16) uint32_t s_blob[kMaxBlobWords];
  __shared__ __align__(16) Best s_best[L * kBlock];   // [level][thread]: the thread's incumbent (touched by the slow path only)
  __shared__ Best s_red[L][kBlock / 32];
  __shared__ __align__(16) int s_thr[8], s_thrm[8];
  __shared__ unsigned long long s_bar;
  __shared__ uint32_t s_item, s_req, s_last, s_slow;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const size_t blob_stride = blob_stride_words(L);
  const uint32_t total_items = a.st->total_items;
  const unsigned long long pio = a.st->per_item_outer;
  if (tid == 0) { mbar_init(&s_bar, 1); s_slow = 0; }
  __syncthreads();
  uint32_t phase = 0;
  long long cur_req = -1;
  unsigned slow_steps = 0;

  for (;;) {
    if (tid == 0) {
      uint32_t it = atomicAdd(&a.st->next_item, 1u);
      // hand-out order: strided across the requests (CallState.perm_sW), so that a request's items do not all start at once
      if (it < total_items) it = (uint32_t)(((unsigned long long)it * a.st->perm_sW) % total_items);
      s_item = it;
      if (it < total_items) {
        // largest r with item_off[r] <= it
        long long lo = 0, hi = a.in.R;
        while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if (a.item_off[mid] <= it) lo = mid; else hi = mid; }
        s_req = (uint32_t)lo;
      }
    }
    __syncthreads();
    const uint32_t item = s_item;
    if (item >= total_items) break;
    const long long r = s_req;
    if (r != cur_req) {
      const uint32_t* gblob = a.blob + (size_t)r * blob_stride;
      if (tid == 0) {
        const int nsp = ((const ReqHdr*)gblob)->nslots_pad;
        const uint32_t bytes = (uint32_t)(kHdrWords + kDem0bWords + nsp * (L + 3)) * 4u;
        tma_load_1d(s_blob, gblob, bytes, &s_bar);
      }
      mbar_wait(&s_bar, phase);
      phase ^= 1;
      cur_req = r;
    }
    const ReqHdr* h = (const ReqHdr*)s_blob;
    int* g_thr = (int*)a.gthr + r * L;
    if (tid < L) {
      const int b = __ldcg(&g_thr[tid]);            // what every block has published so far (bits of a float >= 0)
      s_thr[tid] = b;
      s_thrm[tid] = b > 0 ? b - 1 : (int)0x80000001;  // bits of the float just below it
    }
#pragma unroll
    for (int l = 0; l < L; l++) { Best e; e.C = -1.0f; e.T = INT32_MAX; e.idx = kNoIdx; s_best[l * kBlock + tid] = e; }
    __syncthreads();
    const uint32_t first_item = a.item_off[r];
    const unsigned long long ob = (unsigned long long)(item - first_item) * pio;
    const unsigned long long oe = min(ob + pio, (unsigned long long)h->outer_total);
    const unsigned long long len = oe - ob;
    const unsigned long long per = (len + kBlock - 1) / kBlock;
    const unsigned long long tb = min(ob + (unsigned long long)tid * per, oe);
    const unsigned long long te = min(tb + per, oe);

    if (te > tb) {
      const bool conn = h->conn01 != 0;
      switch (h->K0p) {
        case 2: score_dispatch<L, 2, NB>(conn, s_blob, tb, te - tb, s_thr, s_thrm, s_best + tid, g_thr, &slow_steps); break;
        case 4: score_dispatch<L, 4, NB>(conn, s_blob, tb, te - tb, s_thr, s_thrm, s_best + tid, g_thr, &slow_steps); break;
        case 6: score_dispatch<L, 6, NB>(conn, s_blob, tb, te - tb, s_thr, s_thrm, s_best + tid, g_thr, &slow_steps); break;
        case 8: score_dispatch<L, 8, NB>(conn, s_blob, tb, te - tb, s_thr, s_thrm, s_best + tid, g_thr, &slow_steps); break;
        case 12: score_dispatch<L, 12, NB>(conn, s_blob, tb, te - tb, s_thr, s_thrm, s_best + tid, g_thr, &slow_steps); break;
        default: score_dispatch<L, 16, NB>(conn, s_blob, tb, te - tb, s_thr, s_thrm, s_best + tid, g_thr, &slow_steps); break;
      }
    }
    // ---- block arg-best: warp shuffles, then shared memory, then one record per (item, level) ----
#pragma unroll
    for (int l = 0; l < L; l++) {
      const Best v = warp_best(s_best[l * kBlock + tid]);
      if (lane == 0) s_red[l][wid] = v;
    }
    __syncthreads();
    if (tid < L) {
      Best v = s_red[tid][0];
      for (int w = 1; w < kBlock / 32; w++) { const Best o = s_red[tid][w]; if (better(o.C, o.T, o.idx, v)) v = o; }
      Partial p; p.C = v.C; p.T = v.T; p.idx = v.idx;
      a.partial[(size_t)item * L + tid] = p;
      if (v.idx != kNoIdx) atomicMax(&g_thr[tid], __float_as_int(v.C));
    }
    __syncthreads();
    if (tid == 0) {
      const uint32_t n_it = a.item_off[r + 1] - first_item;
      __threadfence();   // release in the ticket-taking thread, after the block barrier (cumulative over the records above)
      const uint32_t t = atomicAdd(&a.done[r], 1u);
      s_last = (t == n_it - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last) {
      // ---- last block of this request: reduce its items' records and emit the bundle (fused K_final) ----
      __threadfence();
      const uint32_t n_it = a.item_off[r + 1] - first_item;
#pragma unroll
      for (int l = 0; l < L; l++) {
        Best v; v.C = -1.0f; v.T = INT32_MAX; v.idx = kNoIdx;
        for (uint32_t j = tid; j < n_it; j += kBlock) {
          const Partial* pp = &a.partial[(size_t)(first_item + j) * L + l];
          const float4 raw = __ldcg((const float4*)pp);
          Best o; o.C = raw.x; o.T = __float_as_int(raw.y);
          o.idx = ((unsigned long long)__float_as_uint(raw.w) << 32) | (unsigned long long)__float_as_uint(raw.z);
          if (better(o.C, o.T, o.idx, v)) v = o;
        }
        v = warp_best(v);
        if (lane == 0) s_red[l][wid] = v;
      }
      __syncthreads();
      if (tid < L) {
        Best v = s_red[tid][0];
        for (int w = 1; w < kBlock / 32; w++) { const Best o = s_red[tid][w]; if (better(o.C, o.T, o.idx, v)) v = o; }
        emit_record(a, h, r, tid, v);
      }
    }
    __syncthreads();
  }
  if (slow_steps) atomicAdd(&s_slow, slow_steps);
  __syncthreads();
  if (tid == 0 && s_slow) atomicAdd(&a.st->slow_steps, (unsigned long long)s_slow);
}

}  // namespace dyplan

// ---- per-L translation unit body ----------------------------------------------------------------------------------
#ifdef DYPLAN_SCORE_L
namespace dyplan {
#define DYPLAN_CAT2(a, b) a##b
#define DYPLAN_CAT(a, b) DYPLAN_CAT2(a, b)
cudaError_t DYPLAN_CAT(launch_score_l, DYPLAN_SCORE_L)(const CallArgs& a, int nb_class, int grid, cudaStream_t s) {
  constexpr int L = DYPLAN_SCORE_L;
  switch (nb_class) {
    case 0: k_score<L, 0><<<grid, kBlock, 0, s>>>(a); break;
    case 2: k_score<L, 2><<<grid, kBlock, 0, s>>>(a); break;
    case 4: k_score<L, 4><<<grid, kBlock, 0, s>>>(a); break;
    default: k_score<L, 8><<<grid, kBlock, 0, s>>>(a); break;
  }
  return cudaGetLastError();
}
int DYPLAN_CAT(score_occupancy_l, DYPLAN_SCORE_L)(int nb_class) {
  constexpr int L = DYPLAN_SCORE_L;
  int n = 0;
  cudaError_t e;
  switch (nb_class) {
    case 0: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_score<L, 0>, kBlock, 0); break;
    case 2: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_score<L, 2>, kBlock, 0); break;
    case 4: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_score<L, 4>, kBlock, 0); break;
    default: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_score<L, 8>, kBlock, 0); break;
  }
  return e == cudaSuccess ? n : -1;
}
}  // namespace dyplan
#endif
