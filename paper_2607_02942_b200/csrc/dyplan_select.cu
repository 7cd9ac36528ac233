// dyplan_select.cu -- K_select: stateless variant re-scoring under one live pressure vector (
// PAPER.md:219-231 "selects a prepared variant from live load without invoking the optimizer").
// One thread per request: L stored variants x N nodes of plain DP, nothing to tile.
#include "dyplan_internal.cuh"

namespace dyplan {

__device__ __forceinline__ long long scaled_sel(int tau, int mult) { return ((long long)tau * (long long)mult) / 1000; }

__global__ void __launch_bounds__(128) k_select(SelectArgs a) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const dyplan_batch& b = a.in;
  if (r >= b.R) return;
  const int L = a.L, B = b.B, M = b.M;
  int pick = -1, pf = 0, pT = 0;
  double pC = 0.0;

  // request validation under the live vector (same rules as K_stage, L = 1)
  bool ok = true;
  const int n0 = b.node_off[r], n1 = b.node_off[r + 1], N = n1 - n0;
  if (N < 0 || N > DYPLAN_MAX_NODES || n0 < 0 || n1 > b.NN) ok = false;
  if (ok) {
    unsigned long long s = 1;
    for (int n = 0; n < N && ok; n++) {
      const int ob = b.opt_off[n0 + n], K = b.opt_off[n0 + n + 1] - ob;
      if (K < 1 || K > DYPLAN_MAX_OPTS || ob < 0 || ob + K > b.KK) { ok = false; break; }
      if (s > ((1ull << 60) / (unsigned long long)K)) { ok = false; break; }
      s *= (unsigned long long)K;
    }
  }
  if (ok) {
    for (int bb = 0; bb < B; bb++) ok &= a.live[bb] >= 0;
    ok &= b.slo_us[r] >= 0;
    if (b.cap) for (int bb = 0; bb < B; bb++) ok &= b.cap[r * B + bb] >= 0;
    long long tot = 0, dtot = 0;
    for (int n = 0; n < N && ok; n++) {
      const uint32_t pm = b.pred_mask[n0 + n];
      ok &= (pm >> n) == 0;
      const float v = b.vuln[n0 + n];
      ok &= (v >= 0.0f && v <= 1.0f);
      const int ob = b.opt_off[n0 + n], K = b.opt_off[n0 + n + 1] - ob;
      long long mx = 0, dmx = 0;
      for (int k = 0; k < K && ok; k++) {
        const int o = ob + k;
        ok &= b.lat_us[o] >= 0 && b.demand[o] >= 0;
        const float ac = b.acc[o];
        ok &= (ac >= 0.0f && ac <= 1.0f);
        ok &= b.backend[o] < B && b.model[o] < M;
        if (ok) {
          const long long d = scaled_sel(b.lat_us[o], a.live[b.backend[o]]);
          mx = d > mx ? d : mx;
          dmx = b.demand[o] > dmx ? b.demand[o] : dmx;
        }
      }
      tot += mx; dtot += dmx;
    }
    ok &= tot <= (long long)INT32_MAX && dtot <= (long long)INT32_MAX;
  }

  int pD[DYPLAN_MAX_BACKENDS], pdom = 0;
  for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) pD[i] = 0;
  if (ok) {
    const int slo = b.slo_us[r];
    for (int l = 0; l < L; l++) {
      const long long rec = r * L + l;
      if (a.status[rec] != DYPLAN_ST_OK) continue;
      const uint8_t* ch = a.choice + rec * 16;
      int fin[DYPLAN_MAX_NODES];
      int D[DYPLAN_MAX_BACKENDS], Dm[DYPLAN_MAX_MODELS];
      for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) D[i] = 0;
      for (int i = 0; i < DYPLAN_MAX_MODELS; i++) Dm[i] = 0;
      double c = 1.0;
      int T = 0;
      bool chok = true;
      for (int n = 0; n < N; n++) {
        const int ob = b.opt_off[n0 + n], K = b.opt_off[n0 + n + 1] - ob;
        const int k = ch[n];
        if (k >= K) { chok = false; break; }
        const int o = ob + k;
        const int d = (int)scaled_sel(b.lat_us[o], a.live[b.backend[o]]);
        int start = 0;
        const uint32_t pm = b.pred_mask[n0 + n];
        for (int u = 0; u < n; u++) if ((pm >> u) & 1) start = fin[u] > start ? fin[u] : start;
        fin[n] = start + d;
        T = fin[n] > T ? fin[n] : T;
        c = __dmul_rn(c, __dsub_rn(1.0, __dmul_rn((double)b.vuln[n0 + n], __dsub_rn(1.0, (double)b.acc[o]))));
        D[b.backend[o]] += b.demand[o];
        Dm[b.model[o]] += b.demand[o];
      }
      if (!chok) continue;
      const int f = T <= slo;   // caps are level-independent and held at compile time
      bool take;
      if (pick < 0) take = true;
      else if (f != pf) take = f > pf;
      else if (f) take = (c != pC) ? (c > pC) : (T < pT);
      else take = (T != pT) ? (T < pT) : (c > pC);
      if (take) {
        pick = l; pf = f; pC = c; pT = T;
        for (int i = 0; i < DYPLAN_MAX_BACKENDS; i++) pD[i] = D[i];
        pdom = 0;
        for (int m = 1; m < M; m++) if (Dm[m] > Dm[pdom]) pdom = m;
      }
    }
  }
  a.variant[r] = pick;
  if (a.has_rescored) {
    const dyplan_bundle& o = a.rescored;
    if (pick < 0) {
      o.plan_idx[r] = kNoIdx;
      for (int i = 0; i < 16; i++) o.choice[r * 16 + i] = 0xFF;
      o.corr[r] = -1.0f;
      if (o.corr64) o.corr64[r] = -1.0;
      o.lat[r] = INT32_MAX;
      for (int bb = 0; bb < B; bb++) o.dem[r * B + bb] = 0;
      o.dom_model[r] = 0xFF;
      o.status[r] = ok ? DYPLAN_ST_INFEASIBLE : DYPLAN_ST_INVALID;
    } else {
      const uint8_t* ch = a.choice + (r * L + pick) * 16;
      unsigned long long idx = 0, s = 1;
      for (int n = 0; n < N; n++) {
        idx += (unsigned long long)ch[n] * s;
        s *= (unsigned long long)(b.opt_off[n0 + n + 1] - b.opt_off[n0 + n]);
      }
      o.plan_idx[r] = idx;
      for (int i = 0; i < 16; i++) o.choice[r * 16 + i] = ch[i];
      o.corr[r] = (float)pC;
      if (o.corr64) o.corr64[r] = pC;
      o.lat[r] = pT;
      for (int bb = 0; bb < B; bb++) o.dem[r * B + bb] = pD[bb];
      o.dom_model[r] = (uint8_t)pdom;
      o.status[r] = pf ? DYPLAN_ST_OK : DYPLAN_ST_INFEASIBLE;
    }
  }
}

// ---- K_switch: the paper's stateful load-driven selector, one thread per request.  The rule is
// spelled out in include/dyplan.h (dyplan_switch); nothing here solves anything: it reads L records per request. ----
__global__ void __launch_bounds__(128) k_switch(SwitchArgs a) {
  const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const dyplan_batch& b = a.in;
  if (r >= b.R) return;
  const int L = a.L, M = b.M;
  const dyplan_bundle& v = a.bundle;
  const long long rec0 = r * L;
  const int cur = a.cur_variant[r];
  int pick = cur;
  int how = 0;
  auto okv = [&](int k) { return v.status[rec0 + k] == DYPLAN_ST_OK && v.dom_model[rec0 + k] < M; };
  auto qual = [&](int k) { return v.corr64 ? v.corr64[rec0 + k] : (double)v.corr[rec0 + k]; };
  auto load = [&](int k) { return a.model_load[v.dom_model[rec0 + k]]; };
  if (cur < 0 || cur >= L || !okv(cur)) {
    pick = -1;
    for (int k = 0; k < L; k++) if (okv(k)) { pick = k; how = 3; break; }
  } else {
    const float dwell = a.since_switch[r];
    const float lc = load(cur);
    const double qc = qual(cur);
    if (dwell >= a.p.min_dwell && lc == lc) {   // NaN dwell or load: retain
      if (lc > a.p.hi_load) {
        const int dc = v.dom_model[rec0 + cur];
        for (int k = cur + 1; k < L; k++) {
          if (!okv(k)) continue;
          if (v.dom_model[rec0 + k] == dc) continue;          // the same congested class
          const float lk = load(k);
          if (!(lk <= a.p.hi_load)) continue;                   // itself overloaded (or NaN)
          if (!((double)lk <= (double)lc - (double)a.p.load_margin)) continue;   // not sufficiently less loaded
          if (!(qc - qual(k) <= (double)a.p.quality_tol)) continue;
          pick = k; how = 1;
          break;
        }
      } else {
        for (int k = 0; k < cur; k++) {
          if (!okv(k)) continue;
          if (!(load(k) < a.p.lo_load)) continue;
          if (!(qc - qual(k) <= (double)a.p.quality_tol)) continue;
          pick = k; how = 2;
          break;
        }
      }
    }
  }
  if (pick != cur && pick >= 0) {
    // node-boundary safe point: only undispatched nodes take the selected variant's bindings
    const uint32_t dm = a.dispatched[r];
    const int N = b.node_off[r + 1] - b.node_off[r];
    const uint8_t* ch = v.choice + (rec0 + pick) * 16;
    for (int n = 0; n < 16; n++)
      if (n < N && !((dm >> n) & 1)) a.active_choice[r * 16 + n] = ch[n];
  }
  a.cur_variant[r] = pick;
  a.switched[r] = (uint8_t)(pick != cur ? how : 0);
}

cudaError_t launch_switch(const SwitchArgs& a, cudaStream_t s) {
  const unsigned grid = (unsigned)((a.in.R + 127) / 128);
  if (grid == 0) return cudaSuccess;
  k_switch<<<grid, 128, 0, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_select(const SelectArgs& a, cudaStream_t s) {
  const unsigned grid = (unsigned)((a.in.R + 127) / 128);
  if (grid == 0) return cudaSuccess;
  k_select<<<grid, 128, 0, s>>>(a);
  return cudaGetLastError();
}

}  // namespace dyplan
