/* dyplan_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, obviously-correct CPU brute force of what the dyplan hot path computes
 * (definitions C.1 1-11, restated in DESIGN.md section 3).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or call
 * this file.  It shares no code, header, table or constant with paper_2607_02942_b200/csrc/.
 *
 * The method is an exact optimisation, and the CUDA path reaches exactly the brute-force result, so
 * the oracle is the definition written out: enumerate every plan by its canonical index, decode the
 * digits with % and /, score the plan from scratch, keep the best under the fixed order.
 *
 *   plan            one implementation per LLM node                PAPER.md:114-121 Eq.(1); Eq.(3) l.1
 *   latency T       longest path of the selected durations,        PAPER.md:180; Eq.(3)
 *                   "a join waits for the last of its predecessors"
 *   error impact    f = v_n * (1 - q)  per node                    PAPER.md:174; PAPER.md:151 (r^ = 1 - q)
 *   correctness     C = prod_n (1 - v_n (1 - a_n))                 BASELINE.json north_star / configs[0] (reading Q2, Q9)
 *   one solve per level, annotated variants                        PAPER.md:209; Alg.1 l.10-15
 *   dominant model  largest share of planned demand                PAPER.md:219 (reading Q13: ties -> lowest id)
 *   suffix problem  committed bindings fixed, U_t re-optimised     PAPER.md:521-530 App. D Eq.(7)
 *   selection       pick a prepared variant from live pressure
 *
 * Arithmetic: fp64 for correctness, int64 for latency and demand.  Pins: tests/test_oracle_pins.py.
 * Parity unpinned: nothing in this file (the constants lambda_f, lambda_c, lambda_ld, beta of the
 * paper's linear objective are not used by this path).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_NODES 16
#define ORC_MAX_OPTS 16
#define ORC_MAX_B 8
#define ORC_MAX_M 8
#define ORC_MAX_L 8

enum { ORC_OK = 0, ORC_INFEASIBLE = 1, ORC_INVALID = 2, ORC_TOO_LARGE = 3 };
enum { ORC_FIXED_IN_PLACE = 0, ORC_RESIDUAL = 1 };

typedef struct {
  int32_t R, B, M;
  const int32_t *node_off;   /* [R+1]  */
  const int32_t *opt_off;    /* [NN+1] */
  const uint32_t *pred_mask; /* [NN]   */
  const float *vuln;         /* [NN]   */
  const int32_t *lat_us;     /* [KK]   */
  const float *acc;          /* [KK]   */
  const int32_t *demand;     /* [KK]   */
  const uint8_t *backend;    /* [KK]   */
  const uint8_t *model;      /* [KK]   */
  const int32_t *slo_us;     /* [R]    */
  const int32_t *cap;        /* [R*B] or NULL */
} orc_batch;

typedef struct {           /* one record per (request, level), index r*L+l */
  uint64_t *plan_idx;      /* UINT64_MAX if none */
  uint8_t *choice;         /* [.*16], 0xFF padding */
  double *corr;            /* -1 if none */
  int64_t *lat;            /* INT32_MAX if none */
  int64_t *dem;            /* [.*B] */
  uint8_t *dom_model;
  uint8_t *status;
  uint64_t *runner_idx;    /* second-best plan under the order; UINT64_MAX if none */
  double *runner_corr;     /* its C; -1 if none */
  uint64_t *n_feasible;    /* number of feasible plans */
} orc_result;

typedef struct { double C; int64_t T; uint64_t idx; int has; } best_t;

/* definition 7: pi > pi' iff C greater, or equal C and T smaller, or both equal and idx smaller */
static int better(double C, int64_t T, uint64_t idx, const best_t *b) {
  if (!b->has) return 1;
  if (C != b->C) return C > b->C;
  if (T != b->T) return T < b->T;
  return idx < b->idx;
}

typedef struct {
  int N;
  int K[ORC_MAX_NODES];
  int o0[ORC_MAX_NODES];     /* first option of node n in the per-option arrays */
  int n0;                    /* first node */
  uint64_t stride[ORC_MAX_NODES];
} req_t;

static int load_req(const orc_batch *b, int r, req_t *q) {
  q->n0 = b->node_off[r];
  q->N = b->node_off[r + 1] - b->node_off[r];
  if (q->N < 0 || q->N > ORC_MAX_NODES) return ORC_INVALID;
  uint64_t s = 1;
  for (int n = 0; n < q->N; n++) {
    q->o0[n] = b->opt_off[q->n0 + n];
    q->K[n] = b->opt_off[q->n0 + n + 1] - q->o0[n];
    if (q->K[n] < 1 || q->K[n] > ORC_MAX_OPTS) return ORC_INVALID;
    q->stride[n] = s;          /* definition 1: node 0 least significant */
    if (s > (((uint64_t)1 << 60) / (uint64_t)q->K[n])) return ORC_TOO_LARGE;  /* canonical space <= 2^60 */
    s *= (uint64_t)q->K[n];
  }
  return ORC_OK;
}

/* definition 2: d_l(n,k) = floor(tau * mult / 1000) in int64 */
static int64_t scaled(int32_t tau, int32_t mult) { return ((int64_t)tau * (int64_t)mult) / 1000; }

/* Input validation shared by compile/replan/select (SURVEY 8(b) "errors only a device can see"). */
static int validate(const orc_batch *b, int r, const req_t *q, int L, const int32_t *mult /*[L*B]*/) {
  if (b->B < 1 || b->B > ORC_MAX_B || b->M < 1 || b->M > ORC_MAX_M || L < 1 || L > ORC_MAX_L) return ORC_INVALID;
  for (int l = 0; l < L; l++)
    for (int bb = 0; bb < b->B; bb++)
      if (mult[l * b->B + bb] < 0) return ORC_INVALID;
  if (b->slo_us[r] < 0) return ORC_INVALID;
  for (int n = 0; n < q->N; n++) {
    uint32_t pm = b->pred_mask[q->n0 + n];
    if (n < 32 && (pm >> n) != 0) return ORC_INVALID;          /* predecessor must have a smaller index */
    float v = b->vuln[q->n0 + n];
    if (!(v >= 0.0f && v <= 1.0f)) return ORC_INVALID;           /* NaN fails */
    for (int k = 0; k < q->K[n]; k++) {
      int o = q->o0[n] + k;
      if (b->lat_us[o] < 0 || b->demand[o] < 0) return ORC_INVALID;
      if (!(b->acc[o] >= 0.0f && b->acc[o] <= 1.0f)) return ORC_INVALID;
      if (b->backend[o] >= b->B || b->model[o] >= b->M) return ORC_INVALID;
    }
  }
  /* reading Q19: sum_n max_k d_l must fit int32 for every level, and so must sum_n max_k demand */
  for (int l = 0; l < L; l++) {
    int64_t tot = 0;
    for (int n = 0; n < q->N; n++) {
      int64_t mx = 0;
      for (int k = 0; k < q->K[n]; k++) {
        int o = q->o0[n] + k;
        int64_t d = scaled(b->lat_us[o], mult[l * b->B + b->backend[o]]);
        if (d > mx) mx = d;
      }
      tot += mx;
    }
    if (tot > INT32_MAX) return ORC_INVALID;
  }
  int64_t dt = 0;
  for (int n = 0; n < q->N; n++) {
    int64_t mx = 0;
    for (int k = 0; k < q->K[n]; k++)
      if (b->demand[q->o0[n] + k] > mx) mx = b->demand[q->o0[n] + k];
    dt += mx;
  }
  if (dt > INT32_MAX) return ORC_INVALID;
  if (b->cap)
    for (int bb = 0; bb < b->B; bb++)
      if (b->cap[r * b->B + bb] < 0) return ORC_INVALID;
  return ORC_OK;
}

/* Score one plan from scratch (definitions 2-6, 9).  skip_mask: nodes that contribute nothing
 * (RESIDUAL replan, definition 10): duration 0, factor 1, demand 0. */
static void score(const orc_batch *b, const req_t *q, int r, const uint8_t *k, const int32_t *mult /*[B]*/,
                  uint32_t skip_mask, double *C, int64_t *T, int64_t *D /*[B]*/, int *feasible, int *dom) {
  int64_t fin[ORC_MAX_NODES];
  int64_t Dm[ORC_MAX_M];
  double c = 1.0;
  int64_t t = 0;
  for (int bb = 0; bb < b->B; bb++) D[bb] = 0;
  for (int m = 0; m < b->M; m++) Dm[m] = 0;
  for (int n = 0; n < q->N; n++) {
    int o = q->o0[n] + k[n];
    int skip = (skip_mask >> n) & 1;
    int64_t d = skip ? 0 : scaled(b->lat_us[o], mult[b->backend[o]]);
    int64_t start = 0;                                            /* definition 3 */
    uint32_t pm = b->pred_mask[q->n0 + n];
    for (int u = 0; u < n; u++)
      if ((pm >> u) & 1)
        if (fin[u] > start) start = fin[u];
    fin[n] = start + d;
    if (fin[n] > t) t = fin[n];
    if (!skip) {
      c *= 1.0 - (double)b->vuln[q->n0 + n] * (1.0 - (double)b->acc[o]);  /* definition 4, node order */
      D[b->backend[o]] += b->demand[o];                           /* definition 5 */
      Dm[b->model[o]] += b->demand[o];
    }
  }
  int f = t <= (int64_t)b->slo_us[r];                             /* definition 6, inclusive (Q5) */
  if (b->cap)
    for (int bb = 0; bb < b->B; bb++)
      if (D[bb] > (int64_t)b->cap[r * b->B + bb]) f = 0;
  int dm = 0;                                                     /* definition 9, ties -> lowest m */
  for (int m = 1; m < b->M; m++)
    if (Dm[m] > Dm[dm]) dm = m;
  *C = c; *T = t; *feasible = f; *dom = dm;
}

static void write_none(const orc_batch *b, orc_result *out, int rec, int status) {
  out->plan_idx[rec] = UINT64_MAX;
  memset(out->choice + (size_t)rec * 16, 0xFF, 16);
  out->corr[rec] = -1.0;
  out->lat[rec] = INT32_MAX;
  for (int bb = 0; bb < b->B; bb++) out->dem[(size_t)rec * b->B + bb] = 0;
  out->dom_model[rec] = 0xFF;
  out->status[rec] = (uint8_t)status;
  out->runner_idx[rec] = UINT64_MAX;
  out->runner_corr[rec] = -1.0;
  out->n_feasible[rec] = 0;
}

static void decode(const req_t *q, uint64_t idx, uint8_t *k) {
  for (int n = 0; n < q->N; n++) { k[n] = (uint8_t)(idx % (uint64_t)q->K[n]); idx /= (uint64_t)q->K[n]; }
}

/* Brute force for one request: L levels (mult [L*B]) over the plans that agree with `fixed` on the
 * nodes of fixed_mask (compile: fixed_mask = 0).  Writes records rec0 .. rec0+L-1. */
static void solve_request(const orc_batch *b, int r, int L, const int32_t *mult, uint32_t fixed_mask,
                          const uint8_t *fixed /*[N] or NULL*/, uint32_t skip_mask, orc_result *out, int rec0,
                          int inner_parallel) {
  req_t q;
  int st = load_req(b, r, &q);
  if (st == ORC_OK) st = validate(b, r, &q, L, mult);
  if (st == ORC_OK && fixed_mask) {
    if (q.N < 32 && (fixed_mask >> q.N) != 0) st = ORC_INVALID;
    for (int n = 0; n < q.N && st == ORC_OK; n++)
      if ((fixed_mask >> n) & 1) {
        if (fixed[n] >= q.K[n]) st = ORC_INVALID;
        /* reading Q11: the dispatched set is predecessor-closed */
        if ((b->pred_mask[q.n0 + n] & ~fixed_mask) != 0) st = ORC_INVALID;
      }
  }
  /* free nodes and the size of the space that has to be enumerated */
  int nf = 0, fn[ORC_MAX_NODES];
  uint64_t P = 1;
  if (st == ORC_OK) {
    for (int n = 0; n < q.N; n++)
      if (!((fixed_mask >> n) & 1)) { fn[nf++] = n; P *= (uint64_t)q.K[n]; if (P > ((uint64_t)1 << 40)) { st = ORC_TOO_LARGE; break; } }
  }
  if (st != ORC_OK) { for (int l = 0; l < L; l++) write_none(b, out, rec0 + l, st); return; }

  best_t best[ORC_MAX_L], second[ORC_MAX_L];
  uint64_t nfeas[ORC_MAX_L];
  for (int l = 0; l < L; l++) { best[l].has = 0; second[l].has = 0; nfeas[l] = 0; }

  const uint64_t CH = 1 << 14;
  const int64_t nch = (int64_t)((P + CH - 1) / CH);
#pragma omp parallel if (inner_parallel)
  {
    best_t lb[ORC_MAX_L], ls[ORC_MAX_L];
    uint64_t lf[ORC_MAX_L];
    for (int l = 0; l < L; l++) { lb[l].has = 0; ls[l].has = 0; lf[l] = 0; }
#pragma omp for schedule(dynamic, 1)
    for (int64_t ch = 0; ch < nch; ch++) {
      uint64_t j0 = (uint64_t)ch * CH, j1 = j0 + CH < P ? j0 + CH : P;
      for (uint64_t j = j0; j < j1; j++) {
        uint8_t k[ORC_MAX_NODES];
        uint64_t idx = 0, jj = j;
        for (int n = 0; n < q.N; n++) if ((fixed_mask >> n) & 1) k[n] = fixed[n];
        for (int i = 0; i < nf; i++) { int n = fn[i]; k[n] = (uint8_t)(jj % (uint64_t)q.K[n]); jj /= (uint64_t)q.K[n]; }
        for (int n = 0; n < q.N; n++) idx += (uint64_t)k[n] * q.stride[n];   /* definition 1, original radices */
        for (int l = 0; l < L; l++) {
          double C; int64_t T, D[ORC_MAX_B]; int f, dm;
          score(b, &q, r, k, mult + (size_t)l * b->B, skip_mask, &C, &T, D, &f, &dm);
          if (!f) continue;
          lf[l]++;
          if (better(C, T, idx, &lb[l])) { ls[l] = lb[l]; lb[l].C = C; lb[l].T = T; lb[l].idx = idx; lb[l].has = 1; }
          else if (better(C, T, idx, &ls[l])) { ls[l].C = C; ls[l].T = T; ls[l].idx = idx; ls[l].has = 1; }
        }
      }
    }
#pragma omp critical
    {
      for (int l = 0; l < L; l++) {
        nfeas[l] += lf[l];
        /* merge two (best, second) pairs under the total order */
        best_t c[2] = { lb[l], ls[l] };
        for (int i = 0; i < 2; i++) {
          if (!c[i].has) continue;
          if (better(c[i].C, c[i].T, c[i].idx, &best[l])) { second[l] = best[l]; best[l] = c[i]; }
          else if (better(c[i].C, c[i].T, c[i].idx, &second[l])) second[l] = c[i];
        }
      }
    }
  }
  for (int l = 0; l < L; l++) {
    int rec = rec0 + l;
    if (!best[l].has) { write_none(b, out, rec, ORC_INFEASIBLE); continue; }
    uint8_t k[ORC_MAX_NODES];
    decode(&q, best[l].idx, k);
    double C; int64_t T, D[ORC_MAX_B]; int f, dm;
    score(b, &q, r, k, mult + (size_t)l * b->B, skip_mask, &C, &T, D, &f, &dm);
    out->plan_idx[rec] = best[l].idx;
    memset(out->choice + (size_t)rec * 16, 0xFF, 16);
    for (int n = 0; n < q.N; n++) out->choice[(size_t)rec * 16 + n] = k[n];
    out->corr[rec] = C;
    out->lat[rec] = T;
    for (int bb = 0; bb < b->B; bb++) out->dem[(size_t)rec * b->B + bb] = D[bb];
    out->dom_model[rec] = (uint8_t)dm;
    out->status[rec] = ORC_OK;
    out->runner_idx[rec] = second[l].has ? second[l].idx : UINT64_MAX;
    out->runner_corr[rec] = second[l].has ? second[l].C : -1.0;
    out->n_feasible[rec] = nfeas[l];
  }
}

/* ---- exported entry points (host pointers everywhere) ---------------------------------------- */

/* Alg. 1 l.10-15: one exhaustive solve per level; requests r_begin..r_end-1 (others untouched). */
int orc_compile(const orc_batch *b, int L, const int32_t *mult_pm, int r_begin, int r_end, orc_result *out) {
  if (!b || !mult_pm || !out || L < 1 || L > ORC_MAX_L) return -1;
  int nreq = r_end - r_begin;
  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#endif
  if (nreq >= 4 * nthreads) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = r_begin; r < r_end; r++) solve_request(b, r, L, mult_pm, 0, NULL, 0, out, r * L, 0);
  } else {
    for (int r = r_begin; r < r_end; r++) solve_request(b, r, L, mult_pm, 0, NULL, 0, out, r * L, 1);
  }
  return 0;
}

/* App. D Eq.(7): re-optimise the undispatched nodes; one live multiplier vector per query (L = 1). */
int orc_replan(const orc_batch *b, const uint32_t *dispatched_mask, const uint8_t *fixed_choice,
               const int32_t *live_mult_pm /*[R*B]*/, uint32_t flags, int r_begin, int r_end, orc_result *out) {
  if (!b || !dispatched_mask || !fixed_choice || !live_mult_pm || !out) return -1;
  int nreq = r_end - r_begin;
  int nthreads = 1;
#ifdef _OPENMP
  nthreads = omp_get_max_threads();
#endif
  int outer = nreq >= 4 * nthreads;
#pragma omp parallel for schedule(dynamic, 1) if (outer)
  for (int r = r_begin; r < r_end; r++) {
    uint32_t skip = (flags & ORC_RESIDUAL) ? dispatched_mask[r] : 0;
    solve_request(b, r, 1, live_mult_pm + (size_t)r * b->B, dispatched_mask[r], fixed_choice + b->node_off[r],
                  skip, out, r, !outer);
  }
  return 0;
}

/* oracle_score(r, mult, choice): (C, T, D_b, feasible, dominant model) of any plan. Returns status. */
int orc_score(const orc_batch *b, int r, const int32_t *mult_pm /*[B]*/, const uint8_t *choice, uint32_t skip_mask,
              double *C, int64_t *T, int64_t *D, int32_t *feasible, int32_t *dom, uint64_t *idx) {
  req_t q;
  int st = load_req(b, r, &q);
  if (st == ORC_OK) st = validate(b, r, &q, 1, mult_pm);
  if (st != ORC_OK) return st;
  uint64_t id = 0;
  for (int n = 0; n < q.N; n++) {
    if (choice[n] >= q.K[n]) return ORC_INVALID;
    id += (uint64_t)choice[n] * q.stride[n];
  }
  int f, dm;
  score(b, &q, r, choice, mult_pm, skip_mask, C, T, D, &f, &dm);
  *feasible = f; *dom = dm; *idx = id;
  return ORC_OK;
}

/* Definition 11 (S8): re-score the stored variants of each request under ONE live multiplier vector
 * and return the variant index by (feasible desc; C desc, T' asc, l asc); if no stored variant is
 * feasible: (T' asc, C desc, l asc); -1 if the bundle holds no plan for the request.
 * choice: [R*L*16] from a compile; status: [R*L].  Also returns the re-scored T' and C of the pick. */
int orc_select(const orc_batch *b, int L, const uint8_t *choice, const uint8_t *status, const int32_t *live_mult_pm,
               int32_t *variant, int64_t *lat_out, double *corr_out, uint8_t *feasible_out) {
  if (!b || !choice || !status || !live_mult_pm || !variant) return -1;
  for (int r = 0; r < b->R; r++) {
    req_t q;
    variant[r] = -1;
    if (lat_out) lat_out[r] = INT32_MAX;
    if (corr_out) corr_out[r] = -1.0;
    if (feasible_out) feasible_out[r] = 0;
    int st = load_req(b, r, &q);
    if (st == ORC_OK) st = validate(b, r, &q, 1, live_mult_pm);
    if (st != ORC_OK) continue;
    int pick = -1, pf = 0; double pC = 0; int64_t pT = 0;
    for (int l = 0; l < L; l++) {
      int rec = r * L + l;
      if (status[rec] != ORC_OK) continue;
      double C; int64_t T, D[ORC_MAX_B]; int f, dm;
      score(b, &q, r, choice + (size_t)rec * 16, live_mult_pm, 0, &C, &T, D, &f, &dm);
      /* caps are level-independent and held at compile time; feasibility here is the SLO under the live vector */
      f = T <= (int64_t)b->slo_us[r];
      int take;
      if (pick < 0) take = 1;
      else if (f != pf) take = f > pf;
      else if (f) take = (C != pC) ? (C > pC) : (T < pT);      /* equal (C,T): keep the lower l */
      else take = (T != pT) ? (T < pT) : (C > pC);
      if (take) { pick = l; pf = f; pC = C; pT = T; }
    }
    variant[r] = pick;
    if (pick >= 0) {
      if (lat_out) lat_out[r] = pT;
      if (corr_out) corr_out[r] = pC;
      if (feasible_out) feasible_out[r] = (uint8_t)pf;
    }
  }
  return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
