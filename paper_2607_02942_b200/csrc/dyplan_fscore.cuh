// dyplan_fscore.cuh -- K_fscore: enumerate + score + arg-best for requests of the fast class,
// one template per padded level count L.  Included by dyplan_fscore_l<L>.cu with DYPLAN_FSCORE_L defined.
//
// Same walk as k_score (dyplan_score.cuh), but
//   * the slack DP of Eq.(3) runs on exact fp32 integers (k_stage admits a request only when every slack, latency
//     and demand sum stays below 2^22), because on sm_100a FADD/FMUL/FFMA issue at 1 warp-instruction/clk/SMSP
//     while IADD3/LOP3/VIADDMNMX/IMAD issue at 0.5 (measured on this B200);
//   * the work item belongs to one WARP, not one block: no block barrier anywhere in the loop;
//   * per (plan, level) the screen is two FMA-pipe instructions and half an ALU-pipe instruction:
//         x = sat(ap1_l - d0[k0][l])          FADD.SAT   1 iff node 0 (hence every node) meets the SLO at level l
//         z = x * P - pred(thr_l)             FFMA       > 0 iff feasible and C32(plan) >= incumbent of level l
//         zmax = max3(zmax, z, z')            FMNMX3     one per two evaluations
//     with P = C1 * f0[k0] (one FMUL per plan; with caps P is also multiplied by x_cap = sat(slackD_g + 1 - dem0[k0]),
//     node 0's options being laid out in one slot group per backend).  A group whose zmax > 0 is re-walked by the
//     exact, warp-cooperative slow path (order 7 with T and the canonical index), which updates the warp's incumbent.
#pragma once
#include "dyplan_common.cuh"

namespace dyplan {

#ifndef CTX_SHARED_MIN_L
#define CTX_SHARED_MIN_L 4
#endif
template <int L>
struct __align__(16) FWarpShared {
  uint32_t blob[kFastBlobWords];   // the request's staged blob (1-D TMA bulk copy)
  Best best[8];                    // the warp's incumbent per level (written by the cooperative slow path only)
  int thr[8];                      // bits of the best C seen so far per level (this warp + what others published)
  float scr[76];                   // slow path: the flagged lane's group state, broadcast through shared memory;
                                   // [36..64]: subtree bounds (DYPLAN_PRUNE_BOUNDS), written once per work item
  float4 ctx[(L >= CTX_SHARED_MIN_L ? L * 32 : 1)];   // (L >= CTX_SHARED_MIN_L) [l][lane] = {X2, Rm3, U1r, A0r}: node-2 context of every lane, written
                                   // by the heavy step and read by each light step (kept out of the register file)
  unsigned long long bar;          // mbarrier of the TMA copy
  const uint32_t* gblob;           // the request's blob in global memory (approx requests: its int32 tables)
};

#ifndef CTX_SHARED_MIN_L
#define CTX_SHARED_MIN_L 4
#endif
// scratch layout of the cooperative slow path
constexpr int kScrC1 = 0, kScrS1 = 1, kScrAp1 = 9, kScrU1 = 17, kScrR2 = 25, kScrIdx = 34;
// subtree bounds: on/off, largest factor of nodes 2, 1, 0, number of (lane, node-2 sweep) pairs skipped in this item
constexpr int kScrBnd = 36, kScrF2 = 37, kScrF1 = 38, kScrF0 = 39, kScrSkip = 40, kScrMx = 44;   // kScrMx: [node 2, 1, 0][8 levels]
// approx requests: the flagged lane's outer digits (16 bytes) and node 2's slot, for the exact integer re-evaluation
constexpr int kScrDig = 68, kScrSlot2 = 72;

// Directed rounding.  The slack DP adds negated durations (stored rounded up) with round-up adds and
// accumulates demands (stored rounded down) with round-down adds.  When every sum stays below 2^23 nothing rounds and
// the slacks, T and the cap tests are exact (ReqHdr.approx = 0); beyond that each slack the screen forms is an UPPER
// bound of the true one, so a feasible plan is never screened out and what passes is verified with integers.
// The exact instantiation (AX = false) uses the plain operations: every value is an integer below 2^23, no rounding
// occurs, and the compiler keeps its freedom to contract them.
template <bool AX> __device__ __forceinline__ float addu(float a, float b) { return AX ? __fadd_ru(a, b) : a + b; }
template <bool AX> __device__ __forceinline__ float addd(float a, float b) { return AX ? __fadd_rd(a, b) : a + b; }
template <bool AX> __device__ __forceinline__ float subu(float a, float b) { return AX ? __fsub_ru(a, b) : a - b; }
template <bool AX> __device__ __forceinline__ float fmau(float a, float b, float c) { return AX ? __fmaf_ru(a, b, c) : fmaf(a, b, c); }
template <bool AX> __device__ __forceinline__ float addu_sat(float a, float b) {
  if (!AX) return __saturatef(a + b);
  float r;
  asm("add.rp.sat.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
  return r;
}

// Exact re-evaluation of one plan at one level from the int32 tables of an `approx` request: slack DP of Eq.(3) over
// all nodes and per-backend demand sums, as plain integers.  The plan: outer digits and node 2's slot from the flagged
// lane's scratch, node 1's and node 0's slots given.  Returns feasibility; *T_out = critical-path latency.
template <int L>
__device__ __forceinline__ bool exact_check(const FWarpShared<L>* __restrict__ ws, int slot1, int slot0, int l, int* T_out) {
  const uint32_t* sb = ws->blob;
  const ReqHdr* h = (const ReqHdr*)sb;
  const int nsp = h->nslots_pad, Np = h->n_int;
  const int* ilat = (const int*)(ws->gblob + h->ioff);   // [slot][L], global memory (rarely read)
  const int* idem = ilat + nsp * L;                      // [slot]
  const int* s_be = (const int*)(sb + kHdrWords) + nsp * (L + 2);
  const unsigned char* sdig = (const unsigned char*)&ws->scr[kScrDig];
  const int slo = h->slo_c;
  int u[16], D[8];
#pragma unroll
  for (int b = 0; b < 8; b++) D[b] = 0;
  int ms = slo;
  for (int i = Np - 1; i >= 0; --i) {
    const int slot = i >= 3 ? h->optbase[i] + sdig[i] : (i == 2 ? ((const int*)ws->scr)[kScrSlot2] : (i == 1 ? slot1 : slot0));
    int m = slo;
    for (uint32_t dm = h->deps[i]; dm; dm &= dm - 1) m = min(m, u[__ffs(dm) - 1]);
    const int v = m - ilat[slot * L + l];
    u[i] = v;
    ms = min(ms, v);
    const int be = s_be[slot] & 7, dmd = idem[slot];
#pragma unroll
    for (int b = 0; b < 8; b++) D[b] += (b == be) ? dmd : 0;
  }
  bool ok = ms >= 0;
#pragma unroll
  for (int b = 0; b < 8; b++) ok = ok && D[b] <= h->cap[b];
  *T_out = slo - ms;
  return ok;
}

// Loop nest of one lane over `steps` outer indices (digits of internal nodes >= 2, odometer order).  Every lane of
// the warp runs the same number of steps (a lane whose own range is shorter keeps walking with C = 0, which can
// never produce a candidate), so the warp stays converged and the slow path can be cooperative:
//   heavy step  (a digit >= 3 changed)  slack DP of nodes top..3 over local-memory arrays, node-2 context
//   light step  (digit 2)               u2, running minimum, inputs of the middle loop, C2, cap slack; thresholds
//                                       refreshed from what every warp of the request published in g_thr
//   middle loop (digit 1)               ap1_l = min(A0q1_l, (U1_l + 1 - d1_l) * S01): slack bound (+1) of node 0
//   inner block (digit 0, unrolled)     the screen; tables in registers
//   slow path   (any lane saw z > 0)    for each flagged lane: its group state goes to shared memory, the 32 lanes
//                                       re-evaluate the K0P x L (plan, level) pairs one per lane with the exact
//                                       order 7 (T and the canonical index), candidates update the warp's incumbent
// AX: the request is `approx` (the integer verification is compiled in; it costs the exact instantiation's enumeration
// loop 6 % through register allocation when present, hence a template parameter and not a run-time test).
template <int L, int K0P, int NB, bool AX>
__device__ __noinline__ void frange(FWarpShared<L>* __restrict__ ws, unsigned long long o_begin, unsigned long long my_count,
                                    unsigned long long steps, int* g_thr, const int Lr, unsigned* __restrict__ slow_io) {
  constexpr int NBX = NB ? NB : 1;
  constexpr int G = NB ? K0P / NB : K0P;
  const int lane = threadIdx.x & 31;
  const uint32_t* sb = ws->blob;
  int* w_thr = ws->thr;
  unsigned slow_steps = 0;
  const ReqHdr* h = (const ReqHdr*)sb;
  const int nsp = h->nslots_pad;
  const float* s_nlat = (const float*)(sb + kHdrWords);   // [slot][L], negated durations
  const float* s_f = s_nlat + nsp * L;
  const float* s_dem = s_f + nsp;
  const int* s_be = (const int*)(s_dem + nsp);
  const unsigned long long* s_idxc = (const unsigned long long*)(s_be + nsp);
  const float* s_dem1b = (const float*)(s_idxc + nsp);   // [k1][8], caps only
  const int Np = h->n_int, K1 = h->K1, K2 = h->Kp[2];
  const int ob2 = h->optbase[2];
  const float slo = h->slo_f, S01 = h->S01, rS01 = 1.0f / h->S01, big12 = h->big12, big02 = h->big02;
  constexpr bool approx = AX;
  const uint32_t deps0 = h->deps[0], deps1 = h->deps[1], deps2 = h->deps[2];

  // inner tables in registers
  float nd0[K0P][L], f0[K0P], ndem0[K0P];
#pragma unroll
  for (int k = 0; k < K0P; k++) {
#pragma unroll
    for (int l = 0; l < L; l++) nd0[k][l] = s_nlat[k * L + l];
    f0[k] = s_f[k];
    ndem0[k] = NB ? -s_dem[k] : 0.0f;
  }
  float capf[NBX];
#pragma unroll
  for (int b = 0; b < NBX; b++) capf[b] = h->capf[b];

  // state of the nodes >= 3 (dynamic indexing -> local memory; touched once per K2*K1*K0 plans)
  float u[16][L];
  float Rm[17][L];
  float Cp[17];
  float Dp[17][NBX];
  unsigned char dig[16];
#pragma unroll
  for (int l = 0; l < L; l++) Rm[Np][l] = slo;
  Cp[Np] = 1.0f;
#pragma unroll
  for (int b = 0; b < NBX; b++) Dp[Np][b] = 0.0f;
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
  bool need_heavy = true;
  constexpr bool kCtxShared = L >= CTX_SHARED_MIN_L;   // many levels: the node-2 context does not fit the register file beside the tables
  float D3[NBX];
  float X2r[L], Rm3r[L], U1rr[L], A0rr[L];   // node-2 context in registers (L < 6)
  float4* cx = ws->ctx + lane;                // this lane's column of the node-2 context in shared memory
  float C3 = 0.0f;
  // Two forms of the screen's incumbent test, same decision up to false positives the slow path rejects:
  //   product form   z = x * (C1 * f0[k0]) - pred(thr_l)            one FMUL per plan
  //   quotient form  z = x * f0[k0] - pred(thr_l) (1 - 2^-20) / C1  one reciprocal and L FMULs per group, none per plan;
  //                  taken when node 0 has more options than that costs.  fl(C1 f0) >= thr implies
  //                  f0 >= thr / (C1 (1 + 2^-24)) > the addend above (reciprocal and products err by < 2^-22), so no
  //                  plan that ties or beats the incumbent is screened out; plans within 1e-6 of it may pass.
  constexpr bool kQuot = K0P >= L + 8;   // (measured: no gain at 8 options x 4 levels, 3 % at 12 x 1)
  float nthrm[L];   // -pred(thr_l) (times 1 - 2^-20 in the quotient form): the screen's addend
  // lane l < Lr reads the bits of the best C the request's warps have published for level l, one light step ahead
  const int* gaddr = g_thr + (lane < Lr ? lane : 0);
  asm volatile("" : "+l"(gaddr));   // keep the address in its own register pair (not rematerialised into a scratch pair)
  int gpub = 0;
  for (unsigned long long step = 0; step < steps; step++) {
    if (need_heavy) {
    need_heavy = false;
    // ---- heavy step ----
    for (int i = top; i >= 3; --i) {
      const int slot = h->optbase[i] + dig[i];
      float m[L];
#pragma unroll
      for (int l = 0; l < L; l++) m[l] = slo;
      for (uint32_t dm = h->deps[i]; dm; dm &= dm - 1) {
        const int j = __ffs(dm) - 1;
#pragma unroll
        for (int l = 0; l < L; l++) m[l] = fminf(m[l], u[j][l]);
      }
#pragma unroll
      for (int l = 0; l < L; l++) {
        const float v = addu<AX>(m[l], s_nlat[slot * L + l]);
        u[i][l] = v;
        Rm[i][l] = fminf(Rm[i + 1][l], v);
      }
      Cp[i] = Cp[i + 1] * s_f[slot];
      if (NB) {
        const int be = s_be[slot];
        const float dm = s_dem[slot];
#pragma unroll
        for (int b = 0; b < NBX; b++) Dp[i][b] = addd<AX>(Dp[i + 1][b], be == b ? dm : 0.0f);
      }
    }
    // ---- subtree bound (DYPLAN_PRUNE_BOUNDS; items whose lanes are in phase, so these branches are warp-uniform) ----
    // Every plan below this prefix has C32 <= ub (rounding is monotone and the factors are taken in the scorer's
    // order); it misses the SLO at level l if a node >= 3 already does, and breaks a cap if the outer nodes' demand
    // already does.  The slow path admits a plan only with C32 >= thr_l, so a prefix that is dead at every level, in
    // every lane, cannot change an incumbent.
    const bool bnd = ws->scr[kScrBnd] != 0.0f;
    bool bskip = false;
    unsigned lvl_alive = 0u;
    if (bnd) {
      const float ub = __fmul_rn(__fmul_rn(__fmul_rn(Cp[3], ws->scr[kScrF2]), ws->scr[kScrF1]), ws->scr[kScrF0]);
      const int tmine = max(((volatile int*)w_thr)[lane & 7], gpub);
#pragma unroll
      for (int l = 0; l < L; l++) {
        const int tl = __shfl_sync(0xffffffffu, tmine, l);
        if (Rm[3][l] >= 0.0f && ub >= __int_as_float(tl)) lvl_alive |= 1u << l;
      }
      if (NB) {
#pragma unroll
        for (int b = 0; b < NBX; b++) if (!(Dp[3][b] <= capf[b])) lvl_alive = 0u;
      }
      if (!(step < my_count)) lvl_alive = 0u;
      bskip = !__any_sync(0xffffffffu, lvl_alive != 0u);
    }
    if (!bskip) {
    float X2[L], U1r[L], A0r[L];
#pragma unroll
    for (int l = 0; l < L; l++) { X2[l] = slo; U1r[l] = slo; A0r[l] = slo; }
    for (uint32_t dm = deps2; dm; dm &= dm - 1) {
      const int j = __ffs(dm) - 1;
#pragma unroll
      for (int l = 0; l < L; l++) X2[l] = fminf(X2[l], u[j][l]);
    }
    for (uint32_t dm = deps1 & ~7u; dm; dm &= dm - 1) {
      const int j = __ffs(dm) - 1;
#pragma unroll
      for (int l = 0; l < L; l++) U1r[l] = fminf(U1r[l], u[j][l]);
    }
    for (uint32_t dm = deps0 & ~7u; dm; dm &= dm - 1) {
      const int j = __ffs(dm) - 1;
#pragma unroll
      for (int l = 0; l < L; l++) A0r[l] = fminf(A0r[l], u[j][l]);
    }
    if (bnd) {
      // second test, with the context just built: node 2, 1 or 0 misses the SLO even with its shortest option behind
      // the outer nodes alone (X2, U1r, A0r only shrink when inner predecessors are added)
      bool alive = false;
#pragma unroll
      for (int l = 0; l < L; l++) {
        const float* mx = &ws->scr[kScrMx + l];   // largest negated duration of nodes 2, 1, 0 at level l
        alive = alive || (((lvl_alive >> l) & 1u) && addu<AX>(X2[l], mx[0]) >= 0.0f && addu<AX>(U1r[l], mx[8]) >= 0.0f && addu<AX>(A0r[l], mx[16]) >= 0.0f);
      }
      bskip = !__any_sync(0xffffffffu, alive);
    }
    if (!bskip) {
#pragma unroll
    for (int l = 0; l < L; l++) {
      if (kCtxShared) {
        cx[l * 32] = make_float4(X2[l], Rm[3][l], U1r[l], A0r[l]);
      } else {
        X2r[l] = X2[l]; Rm3r[l] = Rm[3][l]; U1rr[l] = U1r[l]; A0rr[l] = A0r[l];
      }
    }
    }
    }
    if (bskip) {
      // no lane of the warp can change an incumbent below this prefix: skip node 2's whole sweep
      const unsigned nlive = __popc(__ballot_sync(0xffffffffu, step < my_count));
      if (lane == 0) ((unsigned*)ws->scr)[kScrSkip] += nlive;
      step += (unsigned long long)(K2 - 1);
      gpub = __ldcg(gaddr);   // keep following what the other warps publish while skipping
      int i = 3;
      for (; i < Np; i++) {
        const int d = dig[i] + 1;
        if (d < h->Kp[i]) { dig[i] = (unsigned char)d; break; }
        dig[i] = 0;
      }
      top = i < Np ? i : Np - 1;
      need_heavy = true;
      continue;
    }
    C3 = Cp[3];
#pragma unroll
    for (int b = 0; b < NBX; b++) D3[b] = Dp[3][b];
    }
    __syncwarp();   // lanes whose heavy step was shorter wait here: the code below runs converged
    {
      // thresholds: this warp's, raised by what the other warps of the request had published one light step ago
      // (the load issued here is consumed at the next step, which keeps its L2 latency off the critical path)
      // (lane l derives level l's addend, the warp reads it by shuffle: one max/decrement/negate instead of L)
      const int t = max(((volatile int*)w_thr)[lane & 7], gpub);
      const float nv = __int_as_float((t > 0 ? t - 1 : 0) | (int)0x80000000) * (kQuot ? 0.99999905f : 1.0f);
#pragma unroll
      for (int l = 0; l < L; l++) nthrm[l] = __shfl_sync(0xffffffffu, nv, l);
      gpub = __ldcg(gaddr);
    }

    // ---- light step: node 2 takes option k2 ----
    const bool live = step < my_count;
    const int slot2 = ob2 + k2;
    float R2[L], U1pS[L], A0q1[L];
    float4 c4v[L];
    if (kCtxShared) {
      // all L loads are issued back to back (program-ordered asm), so their latencies overlap instead of chaining
      // through one reused register quad
#pragma unroll
      for (int l = 0; l < L; l++)
        asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(c4v[l].x), "=f"(c4v[l].y), "=f"(c4v[l].z), "=f"(c4v[l].w) : "r"(smem_u32(cx + l * 32)));
    }
#pragma unroll
    for (int l = 0; l < L; l++) {
      float4 c4;
      if (kCtxShared) c4 = c4v[l]; else c4 = make_float4(X2r[l], Rm3r[l], U1rr[l], A0rr[l]);
      const float u2 = addu<AX>(c4.x, s_nlat[slot2 * L + l]);
      R2[l] = fminf(c4.y, u2);
      const float U1 = fminf(c4.z, addu<AX>(u2, big12));
      const float a0 = fminf(c4.w, addu<AX>(u2, big02));
      A0q1[l] = fminf(addu<AX>(a0, 1.0f), fmau<AX>(R2[l], kBigF, kBigF));   // a node >= 2 misses the SLO  =>  bound <= 0
      U1pS[l] = fmau<AX>(U1, S01, S01);                                      // (U1 + 1) * S01
    }
    const float C2 = live ? C3 * s_f[slot2] : 0.0f;   // a lane past its own range scores nothing
    float sD2[NBX];   // cap slack + 1 before nodes 1 and 0
    if (NB) {
      const int be2 = s_be[slot2];
      const float dm2 = s_dem[slot2];
#pragma unroll
      for (int b = 0; b < NBX; b++) sD2[b] = addu<AX>(subu<AX>(capf[b], addd<AX>(D3[b], be2 == b ? dm2 : 0.0f)), 1.0f);
    }

    float zm = 0.0f, zm2 = 0.0f;   // with caps: two max chains (measured: better with caps, worse without)
    // node 1's options are walked by pointer (factor, [L] durations, [8] per-backend demands): an index loop cost four
    // more ALU-pipe instructions per pair of groups for the address arithmetic (measured: 4.6 % of cfg1's time)
    const float* pf1 = s_f + K0P;
    const float* const pf1_end = pf1 + K1;
    const float* pn1 = s_nlat + K0P * L;
    const float* pd1 = s_dem1b;
#pragma unroll 2
    for (; pf1 != pf1_end; pf1++, pn1 += L, pd1 += 8) {
      float C1 = C2 * pf1[0];
      float s1[NBX];
      if (NB) {
        float smin = kBigF;
#pragma unroll
        for (int b = 0; b < NBX; b++) { s1[b] = subu<AX>(sD2[b], pd1[b]); smin = fminf(smin, s1[b]); }
        C1 *= __saturatef(smin);   // a backend is already over its cap: no plan of this group can be a candidate
      }
      float ap1[L];
#pragma unroll
      for (int l = 0; l < L; l++) ap1[l] = fminf(A0q1[l], fmau<AX>(pn1[l], S01, U1pS[l]));
      // ---- screen: K0P x L evaluations ----
      float zodd = 0.0f;             // odd L: the last level of an even k0 waits for the one of k0 + 1 (one FMNMX3 for both)
      float addend[L];
      if (kQuot) {
        float rc;
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(C1));
#pragma unroll
        for (int l = 0; l < L; l++) addend[l] = (NB && !(C1 > 0.0f)) ? -4.0f : nthrm[l] * rc;   // (C1 = 0: a cap is already exceeded)
      } else {
#pragma unroll
        for (int l = 0; l < L; l++) addend[l] = nthrm[l];
      }
#pragma unroll
      for (int k0 = 0; k0 < K0P; k0++) {
        float P = kQuot ? f0[k0] : C1 * f0[k0];
        if (NB) P *= addu_sat<AX>(s1[k0 / G], ndem0[k0]);
        float z[L];
#pragma unroll
        for (int l = 0; l < L; l++) z[l] = fmaf(addu_sat<AX>(ap1[l], nd0[k0][l]), P, addend[l]);
#pragma unroll
        for (int l = 0; l + 1 < L; l += 2) {
          if (NB && (((l >> 1) + k0) & 1)) zm2 = fmaxf(zm2, fmaxf(z[l], z[l + 1]));
          else zm = fmaxf(zm, fmaxf(z[l], z[l + 1]));
        }
        if (L & 1) {
          if (k0 & 1) { if (NB && (k0 & 2)) zm2 = fmaxf(zm2, fmaxf(zodd, z[L - 1])); else zm = fmaxf(zm, fmaxf(zodd, z[L - 1])); }
          else zodd = z[L - 1];
        }
      }
    }
    // one vote per light step: did any of this lane's K1 x K0P x L evaluations pass the screen?
    unsigned flagged = __ballot_sync(0xffffffffu, fmaxf(zm, zm2) > 0.0f);
    if (__builtin_expect(flagged != 0u, 0)) {
      // ---- cooperative slow path: exact order on the K1 groups of every flagged lane ----
      // (what the other warps have published by now is fetched meanwhile and applied on the way out: many flags
      // are stale-threshold flags, and the next steps should not raise them again)
      const int pub = __ldcg(gaddr);
      while (flagged) {
        const int src = __ffs(flagged) - 1;
        flagged &= flagged - 1;
        if (lane == src) {
          slow_steps++;
          ws->scr[kScrC1] = C2;
#pragma unroll
          for (int b = 0; b < NBX; b++) ws->scr[kScrS1 + b] = NB ? sD2[b] : 0.0f;
#pragma unroll
          for (int l = 0; l < L; l++) {
            ws->scr[kScrAp1 + l] = A0q1[l]; ws->scr[kScrU1 + l] = U1pS[l];
            // R2 is only needed here: with the context in shared memory it is re-derived instead of being kept live
            ws->scr[kScrR2 + l] = kCtxShared ? fminf(cx[l * 32].y, addu<AX>(cx[l * 32].x, s_nlat[slot2 * L + l])) : R2[l];
          }
          if (approx) {   // the exact re-evaluation needs the lane's whole plan prefix
#pragma unroll
            for (int w4 = 0; w4 < 4; w4++)
              ((uint32_t*)ws->scr)[kScrDig + w4] = (uint32_t)dig[4 * w4] | ((uint32_t)dig[4 * w4 + 1] << 8) | ((uint32_t)dig[4 * w4 + 2] << 16) | ((uint32_t)dig[4 * w4 + 3] << 24);
            ((int*)ws->scr)[kScrSlot2] = slot2;
          }
        }
        __syncwarp();
        const float gC2 = ws->scr[kScrC1];
        bool have_idx = false;
        unsigned long long gidx2 = 0;
        for (int k1 = 0; k1 < K1; k1++) {
          const int slot1 = K0P + k1;
          // the group's state, recomputed from the light-step state with the screen's own operations
          float gC1 = __fmul_rn(gC2, s_f[slot1]);
          if (NB) {
            float smin = kBigF;
#pragma unroll
            for (int b = 0; b < NBX; b++) smin = fminf(smin, subu<AX>(ws->scr[kScrS1 + b], s_dem1b[k1 * 8 + b]));
            gC1 = __fmul_rn(gC1, __saturatef(smin));
          }
          for (int e0 = 0; e0 < K0P * L; e0 += 32) {
            const int e = e0 + lane;
            bool cand = false;
            float P = 0.0f;
            int T = 0, l = 0, k0 = 0;
            if (e < K0P * L) {
              k0 = e / L;
              l = e - k0 * L;
              P = __fmul_rn(gC1, s_f[k0]);
              if (NB) P = __fmul_rn(P, addu_sat<AX>(subu<AX>(ws->scr[kScrS1 + k0 / G], s_dem1b[k1 * 8 + k0 / G]), -s_dem[k0]));
              const float u1pS = fmau<AX>(s_nlat[slot1 * L + l], S01, ws->scr[kScrU1 + l]);
              const float t1 = addu<AX>(fminf(ws->scr[kScrAp1 + l], u1pS), s_nlat[e]);   // slack + 1 of node 0's path
              const float ms1 = fminf(fminf(t1, u1pS * rS01), addu<AX>(ws->scr[kScrR2 + l], 1.0f));   // least slack + 1
              // exact requests: every quantity is an integer below 2^23, T is exact.  approx requests: ms1 is an upper
              // bound of the least slack, so this T is a LOWER bound; it is replaced by the exact one below
              T = AX ? (int)fminf(fmaxf(__fsub_rd(__fadd_rd(slo, 1.0f), ms1), 0.0f), 2147483520.0f) : (int)((slo + 1.0f) - ms1);
              // phase 1: feasible, and not worse than the warp's incumbent on (C desc, T asc)
              const float bC = ((volatile float*)&ws->best[l].C)[0];
              const int bT = ((volatile int*)&ws->best[l].T)[0];
              cand = P > 0.0f && t1 >= 1.0f && (P > bC || (P == bC && T <= bT)) && P >= __int_as_float(((volatile int*)w_thr)[l]);
              if (AX && cand) {
                // the conservative test passed: now the plan's exact latency, SLO and caps in integers
                int Tx = 0;
                const bool ok = exact_check<L>(ws, slot1, k0, l, &Tx);
                T = Tx;
                cand = ok && (P > bC || (P == bC && T <= bT));
              }
            }
            unsigned cm = __ballot_sync(0xffffffffu, cand);
            if (cm && !have_idx) {
              // phase 2 needs the canonical index of the flagged lane's prefix (nodes >= 2)
              have_idx = true;
              if (lane == src) {
                unsigned long long idx2 = h->base_idx + s_idxc[slot2];
                for (int i = 3; i < Np; i++) idx2 += s_idxc[h->optbase[i] + dig[i]];
                *(unsigned long long*)&ws->scr[kScrIdx] = idx2;
              }
              __syncwarp();
              gidx2 = *(const unsigned long long*)&ws->scr[kScrIdx];
            }
            const unsigned long long idx = gidx2 + s_idxc[slot1] + s_idxc[k0];
            while (cm) {
              const int c = __ffs(cm) - 1;
              cm &= cm - 1;
              const int cl = __shfl_sync(0xffffffffu, l, c);
              const float cP = __shfl_sync(0xffffffffu, P, c);
              const int cT = __shfl_sync(0xffffffffu, T, c);
              const unsigned long long cidx = __shfl_sync(0xffffffffu, idx, c);
              Best cur;
              cur.C = ((volatile float*)&ws->best[cl].C)[0]; cur.T = ((volatile int*)&ws->best[cl].T)[0];
              cur.idx = ((volatile unsigned long long*)&ws->best[cl].idx)[0];
              if (better(cP, cT, cidx, cur)) {   // warp-uniform
                __syncwarp();
                if (lane == 0) {
                  Best nb; nb.C = cP; nb.T = cT; nb.idx = cidx;
                  ws->best[cl] = nb;
                  const int cb = __float_as_int(cP);
                  if (cb > w_thr[cl]) { w_thr[cl] = cb; if (cl < Lr) atomicMax(&g_thr[cl], cb); }
                }
                __syncwarp();
              }
            }
          }
        }
        __syncwarp();
      }
      if (lane < Lr && pub > ((volatile int*)w_thr)[lane]) w_thr[lane] = pub;
      __syncwarp();
#pragma unroll
      for (int l = 0; l < L; l++) {
        const int t = ((volatile int*)w_thr)[l];
        nthrm[l] = __int_as_float((t > 0 ? t - 1 : 0) | (int)0x80000000) * (kQuot ? 0.99999905f : 1.0f);
      }
    }
    // ---- advance ----
    if (++k2 >= K2) {
      k2 = 0;
      int i = 3;
      for (; i < Np; i++) {
        const int d = dig[i] + 1;
        if (d < h->Kp[i]) { dig[i] = (unsigned char)d; break; }
        dig[i] = 0;
      }
      top = i < Np ? i : Np - 1;   // ran off the request's last outer index (only a lane past its own range does)
      need_heavy = true;
    }
  }
  *slow_io += slow_steps;
}

template <int L>
__global__ void __launch_bounds__(kFastWarps * 32, (L >= 6 ? 3 : 4)) k_fscore(const CallArgs a) {
  __shared__ FWarpShared<L> s_w[kFastWarps];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  FWarpShared<L>* ws = &s_w[wid];
  const int Lr = a.L;                                   // real level count (<= L)
  const size_t blob_stride = blob_stride_words(Lr);
  const uint32_t total_items = a.st->total_items_f;
  const uint32_t rec_base = a.st->total_items;          // partial records of the wide class come first
  const unsigned long long pif = a.st->per_item_outer_f;
  const bool small_call = a.st->small_call_f != 0;
  const uint32_t tail_start = a.st->tail_start_f;
  const uint32_t perm_nA = a.st->perm_nA, perm_sA = a.st->perm_sA, perm_sB = a.st->perm_sB;
  if (lane == 0) mbar_init(&ws->bar, 1);
  __syncwarp();
  uint32_t phase = 0;
  long long cur_req = -1;
  unsigned slow_steps = 0;

  for (;;) {
    uint32_t item = 0;
    if (lane == 0) item = atomicAdd(&a.st->next_item_f, 1u);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= total_items) break;
    // hand-out order: strided over the regular items, then over the tail's small ones (CallState.perm_*)
    item = item < perm_nA ? (uint32_t)(((unsigned long long)item * perm_sA) % perm_nA)
                          : perm_nA + (uint32_t)(((unsigned long long)(item - perm_nA) * perm_sB) % (total_items - perm_nA));
    long long r;
    {   // largest r with item_off_f[r] <= item (every lane searches: uniform, L2-resident)
      long long lo = 0, hi = a.in.R;
      while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if (__ldg(&a.item_off_f[mid]) <= item) lo = mid; else hi = mid; }
      r = lo;
    }
    if (r != cur_req) {
      const uint32_t* gblob = a.blob + (size_t)r * blob_stride;
      __syncwarp();
      if (lane == 0) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const uint32_t words = (uint32_t)__ldg(&((const ReqHdr*)gblob)->blob_words);
        tma_load_1d(ws->blob, gblob, words * 4u, &ws->bar);
      }
      if (lane == 0) ws->gblob = gblob;
      mbar_wait(&ws->bar, phase);
      phase ^= 1;
      cur_req = r;
    }
    const ReqHdr* h = (const ReqHdr*)ws->blob;
    int* g_thr = (int*)a.gthr + r * Lr;
    if (lane < 8) ws->thr[lane] = lane < Lr ? __ldcg(&g_thr[lane]) : 0x40000000;   // padded levels: 2.0f, never admitted
    if (lane < 8) { Best e; e.C = -1.0f; e.T = INT32_MAX; e.idx = kNoIdx; ws->best[lane] = e; }
    __syncwarp();
    const uint32_t first_item = __ldg(&a.item_off_f[r]);
    const unsigned long long pir = fast_item_outer(fast_pif_of(pif, tail_start, r), h->Kp[2], small_call);
    const unsigned long long ob = (unsigned long long)(item - first_item) * pir;
    const unsigned long long oe = min(ob + pir, (unsigned long long)h->outer_total);
    const unsigned long long len = oe - ob;
    // lanes take consecutive sub-ranges of the same length (a multiple of node 2's radix, so that every lane is at
    // the same k2 and the heavy steps coincide); every lane runs `per` steps, the ones past its range score nothing
    const unsigned long long K2u = (unsigned long long)h->Kp[2];
    const unsigned long long per0 = (len + 31) / 32;
    const unsigned long long per = per0 < 2 * K2u ? per0 : ((per0 + K2u - 1) / K2u) * K2u;   // (short ranges: all lanes busy beats lanes in phase)
    const unsigned long long tb = min(ob + (unsigned long long)lane * per, oe);
    const unsigned long long te = min(tb + per, oe);
    {
      // subtree bounds: only when every lane starts a sweep of node 2 at the same step (the bound test votes warp-wide)
      const bool bnd = (a.ctx_flags & DYPLAN_PRUNE_BOUNDS) && ob % K2u == 0 && per % K2u == 0;
      if (lane == 0) {
        ws->scr[kScrBnd] = bnd ? 1.0f : 0.0f;
        ((unsigned*)ws->scr)[kScrSkip] = 0u;
        if (bnd) {
          const float* sf = (const float*)(ws->blob + kHdrWords) + h->nslots_pad * L;
          float m2 = 0.0f, m1 = 0.0f, m0 = 0.0f;
          for (int k = 0; k < h->Kp[2]; k++) m2 = fmaxf(m2, sf[h->optbase[2] + k]);
          for (int k = 0; k < h->K1; k++) m1 = fmaxf(m1, sf[h->K0p + k]);
          for (int k = 0; k < h->K0p; k++) m0 = fmaxf(m0, sf[k]);
          ws->scr[kScrF2] = m2; ws->scr[kScrF1] = m1; ws->scr[kScrF0] = m0;
          const float* sl = (const float*)(ws->blob + kHdrWords);   // [slot][L] negated durations
          for (int l = 0; l < L; l++) {
            float x2 = -kBigF, x1 = -kBigF, x0 = -kBigF;
            for (int k = 0; k < h->Kp[2]; k++) x2 = fmaxf(x2, sl[(h->optbase[2] + k) * L + l]);
            for (int k = 0; k < h->K1; k++) x1 = fmaxf(x1, sl[(h->K0p + k) * L + l]);
            for (int k = 0; k < h->K0p; k++) x0 = fmaxf(x0, sl[k * L + l]);   // (padding slots hold -2^25: never the maximum)
            ws->scr[kScrMx + l] = x2; ws->scr[kScrMx + 8 + l] = x1; ws->scr[kScrMx + 16 + l] = x0;
          }
        }
      }
      __syncwarp();
    }
    {
      const unsigned long long n = te - tb;
      const unsigned long long t0 = n ? tb : 0ull;   // an idle lane walks from outer index 0 (with C = 0)
      switch (h->nbc * 32 + h->K0p) {
#define DYPLAN_FCASE(NB_, K_) case NB_ * 32 + K_: if (h->approx) frange<L, K_, NB_, true>(ws, t0, n, per, g_thr, Lr, &slow_steps); \
                                                  else frange<L, K_, NB_, false>(ws, t0, n, per, g_thr, Lr, &slow_steps); break;
        DYPLAN_FCASE(0, 2) DYPLAN_FCASE(0, 4) DYPLAN_FCASE(0, 6) DYPLAN_FCASE(0, 8) DYPLAN_FCASE(0, 12) DYPLAN_FCASE(0, 16)
        DYPLAN_FCASE(2, 2) DYPLAN_FCASE(2, 4) DYPLAN_FCASE(2, 6) DYPLAN_FCASE(2, 8) DYPLAN_FCASE(2, 12) DYPLAN_FCASE(2, 16)
        DYPLAN_FCASE(3, 6) DYPLAN_FCASE(3, 12)
        DYPLAN_FCASE(4, 4) DYPLAN_FCASE(4, 8) DYPLAN_FCASE(4, 16)
        DYPLAN_FCASE(8, 8) DYPLAN_FCASE(8, 16)
#undef DYPLAN_FCASE
        default: break;   // k_stage never stages another shape for this class
      }
    }
    __syncwarp();
    if (lane == 0 && ((const unsigned*)ws->scr)[kScrSkip])
      atomicAdd(&a.st->bound_skipped, (unsigned long long)((const unsigned*)ws->scr)[kScrSkip] * K2u);
    // ---- the warp's incumbents are the item's records; lane l keeps level l ----
    Best mine; mine.C = -1.0f; mine.T = INT32_MAX; mine.idx = kNoIdx;
    if (lane < Lr) mine = ws->best[lane];
    if (lane < Lr) {
      Partial p; p.C = mine.C; p.T = mine.T; p.idx = mine.idx;
      a.partial[(size_t)(rec_base + item) * Lr + lane] = p;
      if (mine.idx != kNoIdx) atomicMax(&g_thr[lane], __float_as_int(mine.C));
    }
    __syncwarp();
    const uint32_t n_it = __ldg(&a.item_off_f[r + 1]) - first_item;
    uint32_t last = 0;
    if (lane == 0) {
      // release: the lanes' record stores happen-before lane 0's fence (warp barrier), the fence is cumulative at gpu
      // scope and precedes the ticket in the same thread -- the pattern the PTX memory model orders
      __threadfence();
      last = (atomicAdd(&a.done[r], 1u) == n_it - 1) ? 1u : 0u;
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (last) {
      // ---- last warp of this request: reduce its items' records and emit the bundle (fused K_final) ----
      __threadfence();
      if constexpr (L >= 6) {
        // many levels: a lane takes an item and reads the records of all its levels (contiguous: one line for 8 levels,
        // the loads independent), keeping a best per level -- level by level, every line is fetched Lr times with one
        // load in flight, 0.4 ms for the 5 K items of configs[4]'s last request, at the very end of the launch
        Best v[L];
#pragma unroll
        for (int l = 0; l < L; l++) { v[l].C = -1.0f; v[l].T = INT32_MAX; v[l].idx = kNoIdx; }
        for (uint32_t j = lane; j < n_it; j += 32) {
          const float4* pp = (const float4*)&a.partial[(size_t)(rec_base + first_item + j) * Lr];
          float4 raw[L];
#pragma unroll
          for (int l = 0; l < L; l++) if (l < Lr) raw[l] = __ldcg(pp + l);
#pragma unroll
          for (int l = 0; l < L; l++) {
            if (l < Lr) {
              Best o; o.C = raw[l].x; o.T = __float_as_int(raw[l].y);
              o.idx = ((unsigned long long)__float_as_uint(raw[l].w) << 32) | (unsigned long long)__float_as_uint(raw[l].z);
              if (better(o.C, o.T, o.idx, v[l])) v[l] = o;
            }
          }
        }
#pragma unroll
        for (int l = 0; l < L; l++) {
          if (l < Lr) {
            const Best w = warp_best(v[l]);
            if (lane == l) mine = w;
          }
        }
      } else
      for (int l = 0; l < Lr; l++) {
        Best v; v.C = -1.0f; v.T = INT32_MAX; v.idx = kNoIdx;
        // (four loads in flight: a request of a small call is cut into a thousand items and more, and this walk by its
        // last warp, one load at a time, was half of such a call's scoring time)
        for (uint32_t j0 = lane; j0 < n_it; j0 += 128) {
          float4 raw[4];
#pragma unroll
          for (int q = 0; q < 4; q++) {
            const uint32_t j = j0 + 32u * q;
            raw[q] = j < n_it ? __ldcg((const float4*)&a.partial[(size_t)(rec_base + first_item + j) * Lr + l])
                              : make_float4(-1.0f, __int_as_float(INT32_MAX), __uint_as_float(0xffffffffu), __uint_as_float(0xffffffffu));
          }
#pragma unroll
          for (int q = 0; q < 4; q++) {
            Best o; o.C = raw[q].x; o.T = __float_as_int(raw[q].y);
            o.idx = ((unsigned long long)__float_as_uint(raw[q].w) << 32) | (unsigned long long)__float_as_uint(raw[q].z);
            if (better(o.C, o.T, o.idx, v)) v = o;
          }
        }
        v = warp_best(v);
        if (lane == l) mine = v;
      }
      if (lane < Lr) emit_record(a, h, r, lane, mine);
    }
    __syncwarp();
  }
  slow_steps += __shfl_xor_sync(0xffffffffu, slow_steps, 16);
  slow_steps += __shfl_xor_sync(0xffffffffu, slow_steps, 8);
  slow_steps += __shfl_xor_sync(0xffffffffu, slow_steps, 4);
  slow_steps += __shfl_xor_sync(0xffffffffu, slow_steps, 2);
  slow_steps += __shfl_xor_sync(0xffffffffu, slow_steps, 1);
  if (lane == 0 && slow_steps) atomicAdd(&a.st->slow_steps, (unsigned long long)slow_steps);
}

}  // namespace dyplan

// ---- per-L translation unit body ----------------------------------------------------------------------------------
#ifdef DYPLAN_FSCORE_L
namespace dyplan {
#define DYPLAN_CAT2(a, b) a##b
#define DYPLAN_CAT(a, b) DYPLAN_CAT2(a, b)
cudaError_t DYPLAN_CAT(launch_fscore_l, DYPLAN_FSCORE_L)(const CallArgs& a, int grid, cudaStream_t s) {
  k_fscore<DYPLAN_FSCORE_L><<<grid, kFastWarps * 32, 0, s>>>(a);
  return cudaGetLastError();
}
int DYPLAN_CAT(fscore_occupancy_l, DYPLAN_FSCORE_L)() {
  int n = 0;
  const cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_fscore<DYPLAN_FSCORE_L>, kFastWarps * 32, 0);
  return e == cudaSuccess ? n : -1;
}
}  // namespace dyplan
#endif
