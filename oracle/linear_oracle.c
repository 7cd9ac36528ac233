/* linear_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Brute force of the paper's own objective (the "linear mode"), fp64 / int64, written from
 * the definitions.  Shares no code with paper_2607_02942_b200/csrc/ nor with dyplan_oracle.c.
 *
 *   L1  reach weight   rho(n) = 1 + beta*e*(|R(n)|-1)/(|V|-1) for |V| > 1, rho = 1 for a single node; R(n) holds n
 *                      and every node reachable from it
 *   L2  local utility  w(n,k) = rho(n) q - lambda_f v_n (1 - q) - lambda_c c                Eq.(4) PAPER.md:197;
 *                      f = v * r^, r^ = 1 - q
 *   L3  durations      d(n) = tau[n][k_n]; T = longest path of the d(n) through the DAG     Eq.(3)
 *                      D_tau = sum_n d(n) ("counts every LLM node, including nodes outside
 *                      the critical path")
 *   L4  objective      J_L = sum_n w(n,k_n) - lambda_l T - lambda_ld L D_tau                Eq.(4)/(5) PAPER.md:197, 205
 *   L5  one plan per level L_k: the maximiser of J_{L_k}; ties: T ascending, then canonical index ascending
 *                      (the paper is silent on ties; reading Q6 carried over)               Alg.1 l.10-13 PAPER.md:487-492
 * Every node enters the sums; a node with one option (a tool node, "fixed tool quality and cost terms
 * are constants") adds the same constant to every plan and cannot change the choice.
 * The weights lambda_f, lambda_c, lambda_l, lambda_ld, beta and the levels are never printed numerically in the paper
 * (parity unpinned for constants); the pins in tests/test_linear_pins.py fix the formulas.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LN_MAX_NODES 16
#define LN_MAX_L 8

typedef struct {
  int32_t R;
  const int32_t *node_off;   /* [R+1]  */
  const int32_t *opt_off;    /* [NN+1] */
  const uint32_t *pred_mask; /* [NN]   */
  const float *vuln;         /* [NN]   */
  const int32_t *tau;        /* [KK] nominal durations */
  const float *q;            /* [KK] local quality */
  const float *cost;         /* [KK] normalised call cost */
} ln_batch;

typedef struct { double lambda_f, lambda_c, lambda_l, lambda_ld, beta, effort; } ln_params;

typedef struct {             /* one record per (request, level) */
  uint64_t *plan_idx;
  uint8_t *choice;           /* [.*16] */
  double *J;
  int64_t *T;
  int64_t *Dtau;
  double *runner_J;          /* J of the second-best plan under the order; NaN if there is only one plan */
  uint8_t *status;           /* 0 ok, 2 invalid */
} ln_result;

/* L1 */
void ln_reach_weights(int N, const uint32_t *pred_mask, double beta, double effort, double *rho) {
  uint32_t reach[LN_MAX_NODES];
  for (int n = N - 1; n >= 0; n--) {
    reach[n] = 1u << n;
    for (int s = n + 1; s < N; s++)
      if ((pred_mask[s] >> n) & 1) reach[n] |= reach[s];     /* s is a successor of n: everything s reaches, n reaches */
  }
  for (int n = 0; n < N; n++) {
    int cnt = __builtin_popcount(reach[n]);
    rho[n] = (N > 1) ? 1.0 + beta * effort * (double)(cnt - 1) / (double)(N - 1) : 1.0;
  }
}

/* L2-L4 for one plan; k[n] = option of node n */
static void ln_eval(const ln_batch *b, int r, const ln_params *p, const double *rho, const uint8_t *k, double *W, int64_t *T,
                    int64_t *D) {
  const int n0 = b->node_off[r], N = b->node_off[r + 1] - n0;
  int64_t fin[LN_MAX_NODES];
  *W = 0.0; *T = 0; *D = 0;
  for (int n = 0; n < N; n++) {
    const int o = b->opt_off[n0 + n] + k[n];
    const double q = (double)b->q[o], v = (double)b->vuln[n0 + n];
    *W += rho[n] * q - p->lambda_f * v * (1.0 - q) - p->lambda_c * (double)b->cost[o];
    int64_t start = 0;
    for (int u = 0; u < n; u++)
      if ((b->pred_mask[n0 + n] >> u) & 1) start = fin[u] > start ? fin[u] : start;
    fin[n] = start + (int64_t)b->tau[o];
    if (fin[n] > *T) *T = fin[n];
    *D += (int64_t)b->tau[o];
  }
}

static int ln_valid(const ln_batch *b, int r) {
  const int n0 = b->node_off[r], N = b->node_off[r + 1] - n0;
  if (N < 0 || N > LN_MAX_NODES) return 0;
  for (int n = 0; n < N; n++) {
    const int K = b->opt_off[n0 + n + 1] - b->opt_off[n0 + n];
    if (K < 1 || K > 16) return 0;
    if ((b->pred_mask[n0 + n] >> n) != 0) return 0;
    const float v = b->vuln[n0 + n];
    if (!(v >= 0.0f && v <= 1.0f)) return 0;
    for (int k = 0; k < K; k++) {
      const int o = b->opt_off[n0 + n] + k;
      if (b->tau[o] < 0) return 0;
      if (!(b->q[o] >= 0.0f && b->q[o] <= 1.0f)) return 0;
      if (!(b->cost[o] >= 0.0f) || isinf(b->cost[o])) return 0;
    }
  }
  return 1;
}

/* J of a given plan at a given level (used to re-score the CUDA path's choices) */
int ln_score(const ln_batch *b, int r, const ln_params *p, double level, const uint8_t *choice, double *J, int64_t *T,
             int64_t *D) {
  if (!ln_valid(b, r)) return 2;
  const int n0 = b->node_off[r], N = b->node_off[r + 1] - n0;
  for (int n = 0; n < N; n++)
    if (choice[n] >= b->opt_off[n0 + n + 1] - b->opt_off[n0 + n]) return 2;
  double rho[LN_MAX_NODES], W;
  ln_reach_weights(N, b->pred_mask + n0, p->beta, p->effort, rho);
  ln_eval(b, r, p, rho, choice, &W, T, D);
  *J = W - p->lambda_l * (double)*T - p->lambda_ld * level * (double)*D;
  return 0;
}

/* L5: every plan of every request, by canonical index (node 0 least significant) */
int ln_compile(const ln_batch *b, const ln_params *p, int L, const double *levels, ln_result *out) {
  if (!b || !p || !levels || !out || L < 1 || L > LN_MAX_L) return -1;
#pragma omp parallel for schedule(dynamic, 1)
  for (int r = 0; r < b->R; r++) {
    const int n0 = b->node_off[r], N = b->node_off[r + 1] - n0;
    for (int l = 0; l < L; l++) {
      const int rec = r * L + l;
      out->plan_idx[rec] = UINT64_MAX; out->J[rec] = NAN; out->T[rec] = INT32_MAX; out->Dtau[rec] = 0;
      out->runner_J[rec] = NAN; out->status[rec] = 2;
      memset(out->choice + (size_t)rec * 16, 0xFF, 16);
    }
    if (!ln_valid(b, r)) continue;
    double rho[LN_MAX_NODES];
    ln_reach_weights(N, b->pred_mask + n0, p->beta, p->effort, rho);
    uint64_t P = 1;
    int K[LN_MAX_NODES];
    for (int n = 0; n < N; n++) { K[n] = b->opt_off[n0 + n + 1] - b->opt_off[n0 + n]; P *= (uint64_t)K[n]; }
    double bJ[LN_MAX_L], rJ[LN_MAX_L];
    int64_t bT[LN_MAX_L], bD[LN_MAX_L];
    uint64_t bI[LN_MAX_L];
    int has[LN_MAX_L], hasr[LN_MAX_L];
    for (int l = 0; l < L; l++) { has[l] = 0; hasr[l] = 0; }
    for (uint64_t idx = 0; idx < P; idx++) {
      uint8_t k[LN_MAX_NODES];
      uint64_t t = idx;
      for (int n = 0; n < N; n++) { k[n] = (uint8_t)(t % (uint64_t)K[n]); t /= (uint64_t)K[n]; }
      double W; int64_t T, D;
      ln_eval(b, r, p, rho, k, &W, &T, &D);
      for (int l = 0; l < L; l++) {
        const double J = W - p->lambda_l * (double)T - p->lambda_ld * levels[l] * (double)D;
        int better = !has[l] || J > bJ[l] || (J == bJ[l] && (T < bT[l] || (T == bT[l] && idx < bI[l])));
        if (better) {
          if (has[l]) { rJ[l] = bJ[l]; hasr[l] = 1; }
          bJ[l] = J; bT[l] = T; bD[l] = D; bI[l] = idx; has[l] = 1;
        } else if (!hasr[l] || J > rJ[l]) { rJ[l] = J; hasr[l] = 1; }
      }
    }
    for (int l = 0; l < L; l++) {
      const int rec = r * L + l;
      out->status[rec] = 0;
      out->plan_idx[rec] = bI[l]; out->J[rec] = bJ[l]; out->T[rec] = bT[l]; out->Dtau[rec] = bD[l];
      out->runner_J[rec] = hasr[l] ? rJ[l] : NAN;
      uint64_t t = bI[l];
      for (int n = 0; n < N; n++) { out->choice[(size_t)rec * 16 + n] = (uint8_t)(t % (uint64_t)K[n]); t /= (uint64_t)K[n]; }
    }
  }
  return 0;
}
