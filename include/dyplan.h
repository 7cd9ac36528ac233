/* dyplan.h -- C ABI of the B200-native physical-plan compiler hot path ("dyplan").
 *
 * What it computes (citations: PAPER.md:N = line N of the paper text; BJ = BASELINE.json):
 *   A request is a materialised workflow DAG whose LLM nodes each choose one complete implementation
 *   (model x verification policy x backend = one "option") -- PAPER.md:114-121 Eq.(1), Eq.(3) l.1.
 *   For every plan pi (one option per node) and every backend-pressure level l the library evaluates
 *     C(pi)   = prod_n (1 - v_n (1 - a_{n,k_n}))                    impact-weighted error f = v*(1-q),
 *                                                                   PAPER.md:174-176; product form BJ:north_star
 *     T_l(pi) = longest path of the pressure-scaled durations      PAPER.md:180, Eq.(3)
 *               d_l(n,k) = floor(tau_{n,k} * mult[l][backend_{n,k}] / 1000)
 *     D_b(pi) = sum_n demand_{n,k_n} [backend_{n,k_n} = b]          PAPER.md:203-211 (demand annotations)
 *   and keeps, per (request, level), the best plan with T_l <= SLO and D_b <= cap_b under the fixed order
 *   (C descending, T ascending, canonical plan index ascending) -- the pressure-specialised variants of
 *   Algorithm 1, found by exhaustive enumeration instead of K ILP solves.
 *   dyplan_replan does the same over the undispatched nodes only (App. D Eq.(7));
 *   dyplan_select re-scores the stored variants under one live pressure vector and returns the variant
 *   index per request without re-solving.
 *
 * Memory: the dyplan_batch / dyplan_bundle structs live in HOST memory.  In the plain calls every pointer
 *   field is a DEVICE pointer on the ctx's device; in the *_host calls every pointer field is a HOST pointer
 *   (the library stages the copies itself, on `stream`, and returns after the results are in the host buffers).
 *   The caller owns every buffer and keeps it alive until the stream work completes.  The library allocates only
 *   its own scratch inside dyplan_ctx (grown on demand; growing calls cudaMalloc, nothing else synchronises; the
 *   *_host calls also keep a 256 KB pinned staging buffer there).  dyplan_compile_static allocates nothing at all.
 * Streams: `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Plain calls are
 *   asynchronous on it.  A ctx owns one set of scratch: a call issued on another stream than the previous call of the
 *   same ctx first waits, on the device, for that call's work (an event; the host does not block), so calls of one ctx
 *   never overlap -- use one ctx per stream for concurrency.  A ctx is not thread-safe; separate ctxs are independent.
 * Errors: every call returns 0 or a negative DYPLAN_ERR_* code; nothing throws, aborts or prints.  Problems
 *   only a device can see (malformed DAG, out-of-range table entries, NaN, overflow, plan space too large,
 *   dispatched set not predecessor-closed) are reported per request in dyplan_bundle.status; the other requests
 *   of the batch still compile.
 * There is no CPU fallback: without a CUDA device dyplan_create fails with DYPLAN_ERR_CUDA.
 */
#ifndef DYPLAN_H_
#define DYPLAN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* every entry point below is exported from libdyplan.so (the library is built with hidden default visibility) */
#if defined(__GNUC__)
#define DYPLAN_API __attribute__((visibility("default")))
#else
#define DYPLAN_API
#endif

#define DYPLAN_MAX_NODES 16   /* nodes per request                      */
#define DYPLAN_MAX_OPTS 16    /* options per node                       */
#define DYPLAN_MAX_BACKENDS 8
#define DYPLAN_MAX_MODELS 8
#define DYPLAN_MAX_LEVELS 8   /* pressure levels per compile call       */
#define DYPLAN_MAX_PLANS_LOG2 40 /* enumerated plans per request <= 2^40 */

/* return codes */
#define DYPLAN_OK 0
#define DYPLAN_ERR_NULL (-1)   /* a required pointer is NULL                               */
#define DYPLAN_ERR_LIMIT (-2)  /* R, B, M, L, NN or KK outside the limits above / negative  */
#define DYPLAN_ERR_CUDA (-3)   /* a CUDA runtime call failed; see dyplan_last_cuda_error()  */
#define DYPLAN_ERR_ARG (-4)    /* unknown flag bits, inconsistent sizes                     */

/* per-(request, level) status in dyplan_bundle.status */
#define DYPLAN_ST_OK 0         /* a feasible best plan was found                            */
#define DYPLAN_ST_INFEASIBLE 1 /* no plan meets SLO and caps (sentinel outputs)             */
#define DYPLAN_ST_INVALID 2    /* malformed request (sentinel outputs)                      */
#define DYPLAN_ST_TOO_LARGE 3  /* more than 2^40 plans to enumerate (sentinel outputs)      */

/* dyplan_replan flags (reading Q10: both readings of App. D are offered) */
#define DYPLAN_FIXED_IN_PLACE 0u /* dispatched nodes keep their latency, factor and demand (BJ:configs[3])          */
#define DYPLAN_RESIDUAL 1u       /* dispatched nodes contribute d=0, factor 1, demand 0 ("residual makespan T_t starts
                                    from zero on G_t and spans only undispatched work")               */

typedef struct dyplan_ctx dyplan_ctx;

/* A batch of R requests (or replan queries).  The nodes of a request are listed in a topological order
 * (a finite DAG; branches resolved and loops unrolled before submission).  A tool node is a node with
 * one option (fixed duration, no choice).  NN = node_off[R], KK = opt_off[NN]. */
typedef struct {
  int32_t R;                 /* requests, >= 0                                                                */
  int32_t B;                 /* backends, 1..8                                                                */
  int32_t M;                 /* models, 1..8 (annotations only)                                               */
  int32_t NN;                /* total nodes   (= node_off[R]); bounds every per-node array                    */
  int32_t KK;                /* total options (= opt_off[NN]); bounds every per-option array                  */
  const int32_t* node_off;   /* [R+1]  prefix offsets into the per-node arrays; 0 <= N_r <= 16                */
  const int32_t* opt_off;    /* [NN+1] prefix offsets into the per-option arrays; 1 <= K_n <= 16              */
  const uint32_t* pred_mask; /* [NN]   bit p set => local node p precedes node n; requires p < n             */
  const float* vuln;         /* [NN]   vulnerability v_n in [0,1]; NaN is invalid, not zero   */
  const int32_t* lat_us;     /* [KK]   nominal duration tau_{n,k} >= 0, microseconds                         */
  const float* acc;          /* [KK]   a_{n,k} in [0,1], quality of the complete model+verifier pair         */
  const int32_t* demand;     /* [KK]   token demand >= 0                                                     */
  const uint8_t* backend;    /* [KK]   < B                                                                   */
  const uint8_t* model;      /* [KK]   < M                                                                   */
  const int32_t* slo_us;     /* [R]    latency SLO >= 0, inclusive                                           */
  const int32_t* cap;        /* [R*B]  per-backend demand cap >= 0, inclusive; NULL = no caps                */
} dyplan_batch;

/* Result: one record per (request, level) at index rec = r*L + l.  Sentinels when status != OK:
 * plan_idx = UINT64_MAX, choice = 0xFF.., corr = -1, corr64 = -1, lat = INT32_MAX, dem = 0, dom_model = 0xFF. */
typedef struct {
  uint64_t* plan_idx; /* [R*L]    canonical mixed-radix index sum_n k_n prod_{t<n} K_t (node 0 least significant)  */
  uint8_t* choice;    /* [R*L*16] chosen option per node, 0xFF padding                                        */
  float* corr;        /* [R*L]    C(pi) as the scorer computed it (fp32)                                       */
  double* corr64;     /* [R*L]    C(pi) of the chosen plan re-evaluated in fp64, node order; may be NULL       */
  int32_t* lat;       /* [R*L]    T_l(pi), microseconds                                                        */
  int32_t* dem;       /* [R*L*B]  per-backend demand D_b(pi)                                                   */
  uint8_t* dom_model; /* [R*L]    model with the largest planned demand, ties -> lowest id     */
  uint8_t* status;    /* [R*L]    DYPLAN_ST_*                                                                 */
} dyplan_bundle;

/* Context flags (dyplan_set_flags; default 0 = every option of every node is enumerated).
 * DYPLAN_PRUNE_DOMINATED: before enumerating, drop every option that another option of the same node dominates -- at
 *   least as good a factor f, every level's duration no longer, with caps the same backend and no more demand, and
 *   strictly preferred (f larger, or f equal and a lower option index).  Exact: a dropped option is in no best plan under
 *   the fixed order, so results are those of the full enumeration (parity-tested against the unpruned oracle); what
 *   changes is dyplan_stats.plans, which then counts the plans of the pruned space, and the 2^40 limit, which applies
 *   to the pruned space.  Applies to requests the fp32 scorer takes; others are enumerated in full. */
#define DYPLAN_PRUNE_DOMINATED 1u
/* DYPLAN_PRUNE_BOUNDS: while enumerating, skip a whole subtree (all options of the three innermost enumeration digits
 *   below one assignment of the outer nodes) when no plan in it can replace an incumbent: the outer nodes' demand
 *   already exceeds a cap, or at every level either a node misses the SLO even with the shortest options of the inner
 *   nodes (a latency lower bound: durations are >= 0, so the longest path only grows), or the separable upper bound on
 *   C -- the outer nodes' product times the largest factor of each inner node, rounded as the scorer rounds -- is
 *   below the best C already found for that level (second half).
 *   Exact: results are those of the full enumeration (parity-tested against the unpruned oracle).  dyplan_stats.plans
 *   still counts the whole space; dyplan_stats.bound_skipped counts the outer indices that were not walked. */
#define DYPLAN_PRUNE_BOUNDS 2u
/* DYPLAN_NO_SMALL_PATH: by default a call of at most 32 requests hands every request with at most 2^21 (plan, level)
 *   evaluations to a latency-oriented kernel (one admission-time compile: PAPER.md:211) that scores each plan from
 *   scratch in int32 with no incumbent seeds, work items or persistent grid; records are identical.  This flag sends
 *   every request through the batched scorers instead (used by the tests to compare the two paths). */
#define DYPLAN_NO_SMALL_PATH 4u

/* Create / destroy a context on CUDA device `device_ordinal`.  Fails (DYPLAN_ERR_CUDA) without a device. */
DYPLAN_API int dyplan_create(dyplan_ctx** out, int device_ordinal);
DYPLAN_API int dyplan_destroy(dyplan_ctx* ctx);
DYPLAN_API int dyplan_set_flags(dyplan_ctx* ctx, uint32_t flags); /* DYPLAN_ERR_ARG on unknown bits */

/* Algorithm 1 l.10-15 by exhaustive enumeration: best plan per (request, level).
 * mult_pm: [L*B] per-mille latency multipliers >= 0 per (level, backend) -- device pointer (host in *_host). */
DYPLAN_API int dyplan_compile(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult_pm, dyplan_bundle* out,
                   void* stream);

/* App. D Eq.(7): re-optimise the undispatched nodes of each query, committed bindings fixed
 * ("the merge rejects overlap instead of replacing a committed binding": choice[n] == fixed_choice[n]
 * on dispatched nodes).  dispatched_mask [R]: bit n set => local node n already dispatched; must be predecessor-
 * closed, else status INVALID.  fixed_choice [NN]: read where dispatched.  live_mult_pm [R*B]: one
 * live multiplier vector per query.  out holds one record per query (L = 1).  All nodes dispatched => exactly one
 * plan is scored. */
DYPLAN_API int dyplan_replan(dyplan_ctx* ctx, const dyplan_batch* in, const uint32_t* dispatched_mask, const uint8_t* fixed_choice,
                  const int32_t* live_mult_pm, uint32_t flags, dyplan_bundle* out, void* stream);

/* Section 5.1 as a stateless re-scoring: for each request re-score the L stored variants of
 * `bundle` (uses bundle->choice and bundle->status only) under ONE live multiplier vector live_mult_pm [B] and return
 * variant[r] in [0,L), ordered by (SLO-feasible under the live vector first; then C desc, T' asc, l asc; if no stored
 * variant is feasible: T' asc, C desc, l asc); -1 if the bundle holds no plan for the request.  `rescored` (optional,
 * one record per request, L = 1) receives the picked variant re-scored; its status is OK or INFEASIBLE (picked but
 * over the SLO) or the stored error. */
DYPLAN_API int dyplan_select(dyplan_ctx* ctx, const dyplan_batch* in, const dyplan_bundle* bundle, int32_t L,
                  const int32_t* live_mult_pm, int32_t* variant, dyplan_bundle* rescored, void* stream);

/* Section 5.1 as the paper states it, one decision per request, no solver: the STATEFUL selector.
 * Inputs per request: the index of its active variant (cur_variant, -1 = none installed yet), the time since its last
 * switch, its dispatched-node mask and its active assignment; shared: one load figure per MODEL (the runtime
 * "summarizes the load of replicas serving the same model").  The rule, in the paper's order:
 *   - no active variant (or it is not OK in the bundle): install the lowest-index OK variant          -> switched = 3
 *   - since_switch < min_dwell: retain ("a minimum dwell time between switches")         -> switched = 0
 *   - load[dom(cur)] > hi_load: scan the LATER variants in level order; skip a candidate that is not OK, whose
 *     dominant model is the same congested class, or is itself above hi_load; it must be sufficiently less loaded
 *     (load[dom(k)] <= load[dom(cur)] - load_margin) and its estimated quality drop C(cur) - C(k) must not exceed
 *     quality_tol; the FIRST candidate passing both checks is selected              -> switched = 1
 *   - otherwise ("when load subsides"): the lowest-index EARLIER variant whose dominant-model load is below lo_load
 *     and that passes the quality check                                                -> switched = 2
 *   - no eligible transition: the current selection is retained                                       -> switched = 0
 * Applying the selection (Fig. 7(c)): active_choice[n] takes the selected variant's option only for
 * nodes whose bit in dispatched_mask is clear; dispatched nodes keep their binding.  The dominant model of a variant
 * is bundle->dom_model (decided at compile time), its quality estimate bundle->corr64 (corr if NULL).
 * hi_load, lo_load, load_margin, quality_tol, min_dwell are "configured" in the paper and never printed: parameters
 * here.  A NaN load or since_switch retains the selection.  All pointers are DEVICE pointers. */
typedef struct {
  float hi_load;     /* high-load threshold of the active variant's dominant model                      */
  float lo_load;     /* low-load threshold for returning to an earlier variant                          */
  float load_margin; /* comparison rule: a candidate must be at least this much less loaded             */
  float quality_tol; /* largest accepted drop of the estimated quality C                                */
  float min_dwell;   /* minimum time since the request's last switch (same unit as since_switch)       */
} dyplan_switch_params;

DYPLAN_API int dyplan_switch(dyplan_ctx* ctx, const dyplan_batch* in, const dyplan_bundle* bundle, int32_t L,
                  const dyplan_switch_params* params, const float* model_load /*[M]*/, const float* since_switch /*[R]*/,
                  const uint32_t* dispatched_mask /*[R]*/, int32_t* cur_variant /*[R] in/out*/,
                  uint8_t* active_choice /*[R*16] in/out*/, uint8_t* switched /*[R] out*/, void* stream);

/* Coefficient construction, Algorithm 1 l.1-8 and Eq.(2): bind the offline
 * profiles to the candidate implementations of every node, producing the per-node / per-option arrays the compile
 * calls read.  For node n with skill tag s, role rho and fan-in f (the number of predecessor bits), and option k with
 * model m, backend d and verification policy p:
 *     vuln[n]   = psi[role][s][min(f, F-1)]                                       v_n = Psi(role, skill, fan-in)
 *     acc[k]    = quality[s][m][p]                                                q = Q^(s, m, p),
 *     lat_us[k] = rint( 1e6 * sum_a max_j tokens[s][m][p][a][j] / theta_dec[m][d] + tau_pre_us[m][d] )     Eq.(2)
 *                 ("serial stage durations add, a parallel stage contributes its longest nominal call")
 *     cost[k]   = ( sum_a sum_j tokens[s][m][p][a][j] ) / token_norm              "normalized token count across all base
 *                 and verification calls, including those that execute in parallel"
 * tokens = 0 marks an absent call; stage 0 is base generation.  Gated policies carry their expected demand in the
 * profile (App. A).  theta_dec is in tokens per second at the calibration point b_0.  An index out of
 * range (skill, role, model, backend, policy) or a non-positive theta_dec gives vuln = NaN / acc = NaN / lat_us = -1,
 * which the compile calls report as INVALID for that request.  The arrays of `prof` and every other pointer are DEVICE
 * pointers; `prof` itself is a HOST struct.  demand[k] (optional output, may be NULL) = the option's total token count
 * rounded to int32, the per-model demand annotation of PAPER.md:211. */
typedef struct {
  int32_t S, M, P, D;      /* skill classes, models, verification policies, backends                     */
  int32_t A, J;            /* stages per policy (incl. base generation), parallel calls per stage        */
  int32_t ROLES, F;        /* structural roles, fan-in buckets                                           */
  const float* quality;    /* [S*M*P]                                                                    */
  const float* tokens;     /* [S*M*P*A*J] profiled output-token count of call j in stage a               */
  const float* theta_dec;  /* [M*D] calibrated decode rate, tokens/s                                     */
  const float* tau_pre_us; /* [M*D] aggregate prefill-latency correction, microseconds                   */
  const float* psi;        /* [ROLES*S*F]                                                                */
  float token_norm;        /* > 0                                                                        */
} dyplan_profiles;

DYPLAN_API int dyplan_bind(dyplan_ctx* ctx, const dyplan_profiles* prof, int32_t NN, int32_t KK, const int32_t* opt_off /*[NN+1]*/,
                const uint32_t* pred_mask /*[NN]*/, const uint8_t* skill /*[NN]*/, const uint8_t* role /*[NN]*/,
                const uint8_t* model /*[KK]*/, const uint8_t* backend /*[KK]*/, const uint8_t* policy /*[KK]*/,
                float* vuln /*[NN] out*/, float* acc /*[KK] out*/, int32_t* lat_us /*[KK] out*/, float* cost /*[KK] out*/,
                int32_t* demand /*[KK] out or NULL*/, void* stream);

/* The paper's own objective ("linear mode", Eq.(4)/(5)) over the same plan space, by exhaustive
 * enumeration: for every level L_k maximise
 *     J_L(pi) = sum_n [ rho(n) q - lambda_f v_n (1 - q) - lambda_c c ](n, k_n)  -  lambda_l T(pi)  -  lambda_ld L D_tau(pi)
 * with rho(n) = 1 + beta e (|R(n)| - 1) / (|V| - 1) (rho = 1 for one node; R(n) = n and everything reachable from it,
 * PAPER.md:178), T the longest path of the NOMINAL durations tau (Eq.(3); no pressure multipliers here: the paper's
 * levels weight a demand penalty) and D_tau = sum_n tau(n, k_n).  Ties: T ascending, then canonical
 * index ascending.  Reads in->lat_us (tau), in->acc (q), in->vuln (v), in->demand / backend / model (annotations);
 * in->slo_us and in->cap are ignored (the paper's latency charge is soft).  cost: [KK] DEVICE pointer, c >= 0.
 * params and levels are HOST pointers (levels[L], ascending from 0 in the paper; any values in [0, 1e6] accepted, as for
 * the weights).
 * out: one record per (request, level); corr = J as the scorer computed it (fp32), corr64 = J re-evaluated in fp64,
 * lat = T, dem / dom_model as in dyplan_compile.  extra (optional, DEVICE arrays): dtau [R*L] = D_tau of the chosen
 * plan, quality [R*L] = prod_n (1 - v_n (1 - q)) of the chosen plan (the variant's quality estimate dyplan_switch uses).
 * A request whose duration sum exceeds 2^22 (the scorer keeps T and D_tau as exact fp32 integers) or whose plan space
 * exceeds 2^40 gets status TOO_LARGE; malformed requests get INVALID; the rest of the batch still compiles. */
typedef struct {
  float lambda_f, lambda_c, lambda_l, lambda_ld; /* weights of impact-weighted error, call cost, latency, demand */
  float beta, effort;                            /* reach-weight magnitude and effort e in [0,1]                 */
} dyplan_linear_params;

typedef struct {
  int32_t* dtau;   /* [R*L] or NULL */
  double* quality; /* [R*L] or NULL */
} dyplan_linear_extra;

DYPLAN_API int dyplan_compile_linear(dyplan_ctx* ctx, const dyplan_batch* in, const float* cost,
                          const dyplan_linear_params* params, int32_t L, const float* levels, dyplan_bundle* out,
                          const dyplan_linear_extra* extra, void* stream);

/* The compile / replan / select / compile_linear calls with HOST pointers everywhere (batch fields, multipliers, masks,
 * cost, outputs, extras).  The library copies
 * inputs to the device, runs the same kernels and copies the results back, all on `stream`, and returns after a
 * stream synchronise.  h2d_bytes / d2h_bytes (optional) receive the bytes copied.  Calls below 256 KB move through ONE
 * pinned staging buffer owned by the ctx (one copy each way); a compile / replan call whose packed inputs are at most
 * 8 KB -- one admission-time request -- does not use the copy engine at all: the staging kernel fetches the inputs from
 * the pinned buffer itself and the records are stored straight into it (pinned memory is device-visible), so the call is
 * two launches and a synchronise.  The bytes reported are the same either way. */
DYPLAN_API int dyplan_compile_host(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult_pm, dyplan_bundle* out,
                        void* stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes);
DYPLAN_API int dyplan_replan_host(dyplan_ctx* ctx, const dyplan_batch* in, const uint32_t* dispatched_mask,
                       const uint8_t* fixed_choice, const int32_t* live_mult_pm, uint32_t flags, dyplan_bundle* out,
                       void* stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes);
DYPLAN_API int dyplan_compile_linear_host(dyplan_ctx* ctx, const dyplan_batch* in, const float* cost,
                               const dyplan_linear_params* params, int32_t L, const float* levels, dyplan_bundle* out,
                               const dyplan_linear_extra* extra, void* stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes);
DYPLAN_API int dyplan_select_host(dyplan_ctx* ctx, const dyplan_batch* in, const dyplan_bundle* bundle, int32_t L,
                       const int32_t* live_mult_pm, int32_t* variant, dyplan_bundle* rescored, void* stream,
                       uint64_t* h2d_bytes, uint64_t* d2h_bytes);

/* Introspection for the bench and the tests (no device synchronisation unless stated). */
typedef struct {
  uint64_t plans;       /* plans enumerated by the last compile/replan (sum over valid requests)                 */
  uint64_t evals;       /* (plan, level) evaluations = sum_r plans_r * L                                          */
  uint64_t work_items;  /* (request, plan-range) work items the scorer processed                                  */
  uint64_t slow_steps;  /* inner blocks that took the exact (slow) path                                           */
  uint64_t fast_requests; /* requests scored by the fp32 kernel (the others went to the int32 kernel)             */
  int32_t launches;     /* kernels launched by the last call                                                      */
  int32_t sm_count;     /* SMs of the device                                                                      */
  float score_ms;       /* device time of the scoring kernel of the last call (CUDA events on `stream`)           */
  uint64_t bound_skipped; /* outer indices (assignments of all but the two innermost digits) skipped by DYPLAN_PRUNE_BOUNDS */
  uint64_t approx_requests; /* of fast_requests: those whose latency or demand sums exceed 2^22, scored by the fp32 kernel as a
                               conservative screen with every candidate verified in int32 (results identical)          */
  uint64_t small_requests;  /* requests solved by the small-call kernel (calls of at most 32 requests: every request with at
                               most 2^21 (plan, level) evaluations); they are in neither fast_requests nor work_items     */
} dyplan_stats;
/* Synchronises `stream` of the last call, then fills *out. */
DYPLAN_API int dyplan_last_stats(dyplan_ctx* ctx, dyplan_stats* out);

/* M0: the measured issue rate of the instructions the scorers are made of, on
 * THIS device -- the denominator of the path's roofline ("bound": "alu").  For each entry the library runs a kernel
 * of independent dependency chains of that one SASS instruction (or of the scorer's own instruction mix), one block per
 * SM with 8 warps per SMSP, and reports executed warp-instructions per clock per SMSP from clock64() stamps: the median
 * over the SMs (rate), the slowest and fastest SM.  sm_clock_mhz (optional) receives the SM clock the kernels held
 * (cycles of the longest block / CUDA-event time).  `out` is a HOST array of `capacity` entries; *n_out receives the
 * number written (all of them if capacity allows; DYPLAN_ERR_ARG if capacity < 1).  Synchronises `stream`. */
typedef struct {
  char name[64];   /* SASS mnemonic, or "mix: ..." for an instruction mix                           */
  float rate;      /* warp-instructions / clk / SMSP, median over the SMs (1.0 = the issue port)    */
  float rate_min;  /* slowest SM                                                                    */
  float rate_max;  /* fastest SM                                                                    */
} dyplan_issue_rate;
DYPLAN_API int dyplan_measure_issue_rates(dyplan_ctx* ctx, dyplan_issue_rate* out, int32_t capacity, int32_t* n_out,
                               float* sm_clock_mhz, void* stream);

/* dyplan_compile for callers that must not allocate device memory (work under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same kernels, the same records, but every byte of scratch (staged request
 * blobs, work-item offsets, tickets, incumbent thresholds, partial records, call state) is carved from ONE file-scope
 * `static __device__` array of DYPLAN_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library
 * holds until the process exits.  The call allocates nothing: no cudaMalloc / cudaFree / cudaMallocHost, no growth of
 * the ctx's own scratch (which it does not touch), no host heap.  `in`, `mult_pm`, `out`: DEVICE pointers, exactly as
 * in dyplan_compile; the caller owns inputs and outputs.  Asynchronous on `stream`.
 * Limits: 1 <= L <= 8 as everywhere, and R <= DYPLAN_STATIC_MAX_REQUESTS; a larger R returns DYPLAN_ERR_STATIC_LIMIT
 * (nothing is launched, dyplan_last_cuda_error() holds a sentence naming R and the limit).
 * Sharing: the array is ONE per device for the whole process -- every ctx and every call of this entry point uses it,
 * and it keeps the previous call's contents (the kernels reset the counters they need at the start of each call, as
 * they do for the ctx's scratch).  Two calls that OVERLAP on the GPU (different streams, different ctxs, different
 * host threads) RACE on it and give garbage: issue them on one stream, or order them with events.  The library adds no
 * ordering of its own here.  dyplan_last_stats after this call reports `launches` and `sm_count` only.
 * Graph capture: after one call outside capture on the device (it looks up the array's address and the kernels'
 * occupancy), the call only enqueues kernel launches on `stream` and can be captured and replayed. */
#define DYPLAN_STATIC_MAX_REQUESTS 512
#define DYPLAN_STATIC_SCRATCH_BYTES (16u << 20)
#define DYPLAN_ERR_STATIC_LIMIT (-5) /* the call does not fit the static scratch of dyplan_compile_static */
DYPLAN_API int dyplan_compile_static(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult_pm, dyplan_bundle* out,
                          void* stream);

DYPLAN_API const char* dyplan_strerror(int code);
DYPLAN_API const char* dyplan_last_cuda_error(const dyplan_ctx* ctx); /* "" if none */
DYPLAN_API int dyplan_version(void);                            /* major*10000 + minor*100 + patch */

#ifdef __cplusplus
}
#endif
#endif /* DYPLAN_H_ */
