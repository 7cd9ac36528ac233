// dyplan_api.cu -- the C ABI of include/dyplan.h: argument checks, scratch management, kernel sequencing.
// No arithmetic of the method lives here; every step of the path runs in the kernels.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <new>

#include "dyplan_internal.cuh"

namespace dyplan {
cudaError_t launch_score_l1(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l2(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l3(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l4(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l5(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l6(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l7(const CallArgs&, int, int, cudaStream_t);
cudaError_t launch_score_l8(const CallArgs&, int, int, cudaStream_t);
int score_occupancy_l1(int);
int score_occupancy_l2(int);
int score_occupancy_l3(int);
int score_occupancy_l4(int);
int score_occupancy_l5(int);
int score_occupancy_l6(int);
int score_occupancy_l7(int);
int score_occupancy_l8(int);
static const score_launcher_t kLaunch[8] = {launch_score_l1, launch_score_l2, launch_score_l3, launch_score_l4,
                                            launch_score_l5, launch_score_l6, launch_score_l7, launch_score_l8};
cudaError_t launch_fscore_l1(const CallArgs&, int, cudaStream_t);
cudaError_t launch_fscore_l2(const CallArgs&, int, cudaStream_t);
cudaError_t launch_fscore_l3(const CallArgs&, int, cudaStream_t);
cudaError_t launch_fscore_l4(const CallArgs&, int, cudaStream_t);
cudaError_t launch_fscore_l6(const CallArgs&, int, cudaStream_t);
cudaError_t launch_fscore_l8(const CallArgs&, int, cudaStream_t);
int fscore_occupancy_l1();
int fscore_occupancy_l2();
int fscore_occupancy_l3();
int fscore_occupancy_l4();
int fscore_occupancy_l6();
int fscore_occupancy_l8();
// indexed by the real level count - 1 (levels 5 and 7 run in the 6- and 8-level instantiations)
static const fscore_launcher_t kFLaunch[8] = {launch_fscore_l1, launch_fscore_l2, launch_fscore_l3, launch_fscore_l4,
                                              launch_fscore_l6, launch_fscore_l6, launch_fscore_l8, launch_fscore_l8};
typedef int (*focc_fn_t)();
static const focc_fn_t kFOcc[8] = {fscore_occupancy_l1, fscore_occupancy_l2, fscore_occupancy_l3, fscore_occupancy_l4,
                                   fscore_occupancy_l6, fscore_occupancy_l6, fscore_occupancy_l8, fscore_occupancy_l8};
typedef int (*occ_fn_t)(int);
static const occ_fn_t kOcc[8] = {score_occupancy_l1, score_occupancy_l2, score_occupancy_l3, score_occupancy_l4,
                                 score_occupancy_l5, score_occupancy_l6, score_occupancy_l7, score_occupancy_l8};
}  // namespace dyplan

using namespace dyplan;

struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
};

struct dyplan_ctx {
  int device = 0;
  int sm_count = 0;
  cudaError_t last_err = cudaSuccess;
  char errbuf[256] = {0};
  // scratch
  DevBuf blob, item_off, done, gthr, partial, state;   // item_off holds both classes' offset arrays
  DevBuf lin_blob, lin_gj, lin_gkey, lin_misc;          // linear mode
  bool last_linear = false;
  uint32_t flags = 0;
  // staging for the *_host calls: one device arena, one pinned-or-not host side is the caller's
  DevBuf arena;
  void* hstage = nullptr;          // pinned host image of the arena for small *_host calls (one copy in, one copy out)
  size_t hstage_cap = 0;
  // occupancy cache [L-1][nb index]
  int occ[8][4];
  int focc[8];
  // last call
  cudaStream_t last_stream = nullptr;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  cudaEvent_t ev_done = nullptr;   // end of the last call that used the ctx's scratch (ordering across streams)
  cudaStream_t done_stream = nullptr;
  bool have_done = false;
  bool have_events = false;
  int last_launches = 0;
  int last_L = 0;
};

static int fail_cuda(dyplan_ctx* c, cudaError_t e) {
  c->last_err = e;
  snprintf(c->errbuf, sizeof(c->errbuf), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
  return DYPLAN_ERR_CUDA;
}
#define CK(call)                                        \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) return fail_cuda(ctx, e__); \
  } while (0)

static int ensure(dyplan_ctx* ctx, DevBuf& b, size_t bytes) {
  if (bytes <= b.cap) return DYPLAN_OK;
  if (b.p) CK(cudaFree(b.p));
  b.p = nullptr; b.cap = 0;
  size_t want = bytes + bytes / 4 + 256;
  CK(cudaMalloc(&b.p, want));
  b.cap = want;
  return DYPLAN_OK;
}

// The ctx owns ONE set of scratch (staged blobs, counters, partial records, the *_host arena).  Calls on one stream are
// ordered by the stream; a call arriving on ANOTHER stream first waits (on the device) for the previous call's work.
static int order_after_previous(dyplan_ctx* ctx, cudaStream_t stream) {
  if (ctx->have_done && ctx->done_stream != stream) CK(cudaStreamWaitEvent(stream, ctx->ev_done, 0));
  return DYPLAN_OK;
}
static int mark_done(dyplan_ctx* ctx, cudaStream_t stream) {
  CK(cudaEventRecord(ctx->ev_done, stream));
  ctx->done_stream = stream; ctx->have_done = true;
  return DYPLAN_OK;
}

static int nb_index(int nb_class) { return nb_class == 0 ? 0 : nb_class == 2 ? 1 : nb_class == 4 ? 2 : 3; }

extern "C" {

int dyplan_version(void) { return 100; }

const char* dyplan_strerror(int code) {
  switch (code) {
    case DYPLAN_OK: return "ok";
    case DYPLAN_ERR_NULL: return "a required pointer is NULL";
    case DYPLAN_ERR_LIMIT: return "R, B, M, L, NN or KK outside the supported limits";
    case DYPLAN_ERR_CUDA: return "a CUDA runtime call failed (see dyplan_last_cuda_error)";
    case DYPLAN_ERR_ARG: return "invalid argument";
    case DYPLAN_ERR_STATIC_LIMIT: return "the call exceeds the static scratch of dyplan_compile_static (R > DYPLAN_STATIC_MAX_REQUESTS = 512)";
    default: return "unknown error";
  }
}

const char* dyplan_last_cuda_error(const dyplan_ctx* ctx) { return ctx ? ctx->errbuf : ""; }

int dyplan_create(dyplan_ctx** out, int device_ordinal) {
  if (!out) return DYPLAN_ERR_NULL;
  *out = nullptr;
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || device_ordinal < 0 || device_ordinal >= n) return DYPLAN_ERR_CUDA;
  dyplan_ctx* ctx = new (std::nothrow) dyplan_ctx();
  if (!ctx) return DYPLAN_ERR_ARG;
  ctx->device = device_ordinal;
  if (cudaSetDevice(device_ordinal) != cudaSuccess ||
      cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device_ordinal) != cudaSuccess ||
      cudaEventCreate(&ctx->ev0) != cudaSuccess || cudaEventCreate(&ctx->ev1) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_done, cudaEventDisableTiming) != cudaSuccess) {
    delete ctx;
    return DYPLAN_ERR_CUDA;
  }
  for (int i = 0; i < 8; i++) { for (int j = 0; j < 4; j++) ctx->occ[i][j] = 0; ctx->focc[i] = 0; }
  *out = ctx;
  return DYPLAN_OK;
}

int dyplan_set_flags(dyplan_ctx* ctx, uint32_t flags) {
  if (!ctx) return DYPLAN_ERR_NULL;
  if (flags & ~(DYPLAN_PRUNE_DOMINATED | DYPLAN_PRUNE_BOUNDS | DYPLAN_NO_SMALL_PATH)) return DYPLAN_ERR_ARG;
  ctx->flags = flags;
  return DYPLAN_OK;
}

int dyplan_destroy(dyplan_ctx* ctx) {
  if (!ctx) return DYPLAN_ERR_NULL;
  cudaSetDevice(ctx->device);
  DevBuf* bufs[] = {&ctx->blob, &ctx->item_off, &ctx->done, &ctx->gthr, &ctx->partial, &ctx->state, &ctx->arena,
                    &ctx->lin_blob, &ctx->lin_gj, &ctx->lin_gkey, &ctx->lin_misc};
  for (DevBuf* b : bufs) if (b->p) cudaFree(b->p);
  if (ctx->hstage) cudaFreeHost(ctx->hstage);
  if (ctx->ev0) cudaEventDestroy(ctx->ev0);
  if (ctx->ev1) cudaEventDestroy(ctx->ev1);
  if (ctx->ev_done) cudaEventDestroy(ctx->ev_done);
  delete ctx;
  return DYPLAN_OK;
}

}  // extern "C"

static int check_batch(const dyplan_batch* in, bool need_arrays) {
  if (!in) return DYPLAN_ERR_NULL;
  if (in->R < 0 || in->B < 1 || in->B > DYPLAN_MAX_BACKENDS || in->M < 1 || in->M > DYPLAN_MAX_MODELS || in->NN < 0 ||
      in->KK < 0 || in->R > (1 << 24))
    return DYPLAN_ERR_LIMIT;
  if (need_arrays && in->R > 0) {
    if (!in->node_off || !in->opt_off || !in->slo_us) return DYPLAN_ERR_NULL;
    if (in->NN > 0 && (!in->pred_mask || !in->vuln)) return DYPLAN_ERR_NULL;
    if (in->KK > 0 && (!in->lat_us || !in->acc || !in->demand || !in->backend || !in->model)) return DYPLAN_ERR_NULL;
  }
  return DYPLAN_OK;
}

static int check_bundle(const dyplan_bundle* o) {
  if (!o) return DYPLAN_ERR_NULL;
  if (!o->plan_idx || !o->choice || !o->corr || !o->lat || !o->dem || !o->dom_model || !o->status) return DYPLAN_ERR_NULL;
  return DYPLAN_OK;
}

// The plain (device-pointer) calls cannot see the option counts, but the sizes in the struct bound them: a request has
// at most min(NN, 16) nodes, at most KK options in all and at most 16 per node, so at most max_n min(KK / n, 16)^n plans
// (AM-GM; exact for one request with equal counts).  When that bound times L fits k_small's limit, every request that
// k_stage accepts is small, and the batched scorers have nothing to do: their four launches (about 20 us) are not
// issued.  (Taking the maximum over n keeps the bound valid when NN overstates the node count; a KK that understates
// the option count makes k_stage reject the request.)
static bool sizes_prove_all_small(const dyplan_batch* in, int32_t L) {
  if (in->NN <= 0 || in->KK <= 0) return false;
  double worst = 0.0;   // log2 of the bound
  const int nmax = in->NN < DYPLAN_MAX_NODES ? in->NN : DYPLAN_MAX_NODES;
  for (int n = 1; n <= nmax; n++) {
    double k = (double)in->KK / (double)n;
    if (k > (double)DYPLAN_MAX_OPTS) k = (double)DYPLAN_MAX_OPTS;
    if (k < 1.0) k = 1.0;
    const double b = (double)n * log2(k);
    if (b > worst) worst = b;
  }
  return worst + log2((double)L) <= 20.99;
}

// compile and replan share everything but two arguments
// all_small: the caller (a *_host entry point, which sees the option counts) has established that every request of the
// call is one k_small takes, so the batched scorers are not launched at all
static int run_solve(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult, const uint32_t* dispatched,
                     const uint8_t* fixed_choice, uint32_t flags, bool is_replan, dyplan_bundle* out, cudaStream_t stream,
                     bool all_small = false, const void* img_src = nullptr, void* img_dst = nullptr, size_t img_bytes = 0) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = check_batch(in, true);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  if (flags & ~DYPLAN_RESIDUAL) return DYPLAN_ERR_ARG;
  ctx->last_launches = 0;
  ctx->have_events = false;
  ctx->last_stream = stream;
  ctx->last_L = L;
  ctx->last_linear = false;
  if (in->R == 0) return DYPLAN_OK;
  if (!mult) return DYPLAN_ERR_NULL;
  if (is_replan && (!dispatched || (in->NN > 0 && !fixed_choice))) return DYPLAN_ERR_NULL;
  rc = check_bundle(out);
  if (rc) return rc;
  CK(cudaSetDevice(ctx->device));

  if ((rc = order_after_previous(ctx, stream))) return rc;
  const size_t R = (size_t)in->R;
  const int nbc = nb_class_of(in->B, in->cap != nullptr);
  int& occ = ctx->occ[L - 1][nb_index(nbc)];
  if (occ <= 0) {
    occ = kOcc[L - 1](nbc);
    if (occ <= 0) return fail_cuda(ctx, cudaGetLastError() == cudaSuccess ? cudaErrorLaunchOutOfResources : cudaPeekAtLastError());
  }
  int& focc = ctx->focc[L - 1];
  if (focc <= 0) {
    focc = kFOcc[L - 1]();
    if (focc <= 0) return fail_cuda(ctx, cudaGetLastError() == cudaSuccess ? cudaErrorLaunchOutOfResources : cudaPeekAtLastError());
  }
  // persistent grids: every block resident, work pulled from device counters
  const int grid = ctx->sm_count * occ;
  const int fgrid = ctx->sm_count * focc;
  const uint32_t target_items_f = (uint32_t)(fgrid * kFastWarps) * fast_items_per_warp(focc);
  // room for 4x the items aimed at: k_plan cuts the last eighth of the requests into 4x smaller items (a short tail:
  // 1.4x the items when the requests are alike, more when the last ones are the large ones) and checks the exact count
  const uint32_t max_items = (uint32_t)(2 * R + 2) + 2u * (4u * target_items_f > 32768u ? 4u * target_items_f : 32768u);
  if ((rc = ensure(ctx, ctx->blob, R * blob_stride_words(L) * 4))) return rc;
  if ((rc = ensure(ctx, ctx->item_off, 2 * (R + 1) * 4))) return rc;
  if ((rc = ensure(ctx, ctx->done, R * 4))) return rc;
  if ((rc = ensure(ctx, ctx->gthr, R * L * 4))) return rc;
  if ((rc = ensure(ctx, ctx->partial, (size_t)max_items * L * sizeof(Partial)))) return rc;
  if ((rc = ensure(ctx, ctx->state, sizeof(CallState)))) return rc;

  CallArgs a;
  memset(&a, 0, sizeof(a));
  a.in = *in; a.out = *out; a.L = L; a.mult = mult; a.dispatched = dispatched; a.fixed_choice = fixed_choice;
  a.flags = flags; a.is_replan = is_replan ? 1 : 0; a.ctx_flags = ctx->flags;
  a.blob = (uint32_t*)ctx->blob.p; a.item_off = (uint32_t*)ctx->item_off.p; a.item_off_f = a.item_off + (R + 1);
  a.done = (uint32_t*)ctx->done.p; a.target_items_f = target_items_f; a.fast_warps = (uint32_t)(fgrid * kFastWarps);
  a.gthr = (float*)ctx->gthr.p; a.partial = (Partial*)ctx->partial.p; a.st = (CallState*)ctx->state.p;
  a.max_items = max_items;
  a.img_src = (const uint4*)img_src; a.img_dst = (uint4*)img_dst; a.img_vec = (uint32_t)((img_bytes + 15) / 16);
  a.small_mode = (in->R <= kSmallMaxR && !(ctx->flags & DYPLAN_NO_SMALL_PATH)) ? 1 : 0;
  a.small_split = a.small_mode ? (kSmallBlocksPerSm * ctx->sm_count / (int)in->R > 1 ? kSmallBlocksPerSm * ctx->sm_count / (int)in->R : 1) : 1;

  if (a.small_mode && !all_small && sizes_prove_all_small(in, L)) all_small = true;
  CK(launch_stage(a, stream));
  int launches = 1;
  const bool only_small = a.small_mode && all_small;
  // score_ms brackets the scorers: from k_small on in a small call, else the two batched scorers
  if (a.small_mode) { CK(cudaEventRecord(ctx->ev0, stream)); CK(launch_small(a, stream)); launches++; }   // admission path
  if (!only_small) {
    CK(launch_seed(a, stream));
    CK(launch_plan(a, stream));
    if (!a.small_mode) CK(cudaEventRecord(ctx->ev0, stream));
    CK(kFLaunch[L - 1](a, fgrid, stream));      // fp32 scorer: requests of the fast class
    CK(kLaunch[L - 1](a, nbc, grid, stream));   // int32 scorer: the rest (exits at once when it has no work items)
    launches += 4;
  }
  CK(cudaEventRecord(ctx->ev1, stream));
  ctx->have_events = true;
  ctx->last_launches = launches;
  return mark_done(ctx, stream);
}

extern "C" {

int dyplan_compile(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult_pm, dyplan_bundle* out, void* stream) {
  return run_solve(ctx, in, L, mult_pm, nullptr, nullptr, 0, false, out, (cudaStream_t)stream);
}

int dyplan_replan(dyplan_ctx* ctx, const dyplan_batch* in, const uint32_t* dispatched_mask, const uint8_t* fixed_choice,
                  const int32_t* live_mult_pm, uint32_t flags, dyplan_bundle* out, void* stream) {
  return run_solve(ctx, in, 1, live_mult_pm, dispatched_mask, fixed_choice, flags, true, out, (cudaStream_t)stream);
}

int dyplan_select(dyplan_ctx* ctx, const dyplan_batch* in, const dyplan_bundle* bundle, int32_t L, const int32_t* live_mult_pm,
                  int32_t* variant, dyplan_bundle* rescored, void* stream) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = check_batch(in, true);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  ctx->last_launches = 0;
  ctx->have_events = false;
  ctx->last_stream = (cudaStream_t)stream;
  if (in->R == 0) return DYPLAN_OK;
  if (!bundle || !bundle->choice || !bundle->status || !live_mult_pm || !variant) return DYPLAN_ERR_NULL;
  if (rescored && (rc = check_bundle(rescored))) return rc;
  CK(cudaSetDevice(ctx->device));
  SelectArgs a;
  memset(&a, 0, sizeof(a));
  a.in = *in; a.choice = bundle->choice; a.status = bundle->status; a.L = L; a.live = live_mult_pm; a.variant = variant;
  if (rescored) { a.rescored = *rescored; a.has_rescored = 1; }
  CK(launch_select(a, (cudaStream_t)stream));
  ctx->last_launches = 1;
  return DYPLAN_OK;
}

int dyplan_switch(dyplan_ctx* ctx, const dyplan_batch* in, const dyplan_bundle* bundle, int32_t L, const dyplan_switch_params* params,
                  const float* model_load, const float* since_switch, const uint32_t* dispatched_mask, int32_t* cur_variant,
                  uint8_t* active_choice, uint8_t* switched, void* stream) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = check_batch(in, false);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  ctx->last_launches = 0;
  ctx->have_events = false;
  ctx->last_stream = (cudaStream_t)stream;
  if (in->R == 0) return DYPLAN_OK;
  if (!in->node_off || !params || !bundle || !bundle->choice || !bundle->status || !bundle->dom_model ||
      (!bundle->corr64 && !bundle->corr) || !model_load || !since_switch || !dispatched_mask || !cur_variant ||
      !active_choice || !switched)
    return DYPLAN_ERR_NULL;
  if (!(params->hi_load >= params->lo_load) || !(params->load_margin >= 0.0f) || !(params->quality_tol >= 0.0f))
    return DYPLAN_ERR_ARG;
  CK(cudaSetDevice(ctx->device));
  SwitchArgs a;
  memset(&a, 0, sizeof(a));
  a.in = *in; a.bundle = *bundle; a.L = L; a.p = *params; a.model_load = model_load; a.since_switch = since_switch;
  a.dispatched = dispatched_mask; a.cur_variant = cur_variant; a.active_choice = active_choice; a.switched = switched;
  CK(launch_switch(a, (cudaStream_t)stream));
  ctx->last_launches = 1;
  return DYPLAN_OK;
}

int dyplan_bind(dyplan_ctx* ctx, const dyplan_profiles* prof, int32_t NN, int32_t KK, const int32_t* opt_off, const uint32_t* pred_mask,
                const uint8_t* skill, const uint8_t* role, const uint8_t* model, const uint8_t* backend, const uint8_t* policy,
                float* vuln, float* acc, int32_t* lat_us, float* cost, int32_t* demand, void* stream) {
  if (!ctx || !prof) return DYPLAN_ERR_NULL;
  if (NN < 0 || KK < 0) return DYPLAN_ERR_LIMIT;
  if (prof->S < 1 || prof->M < 1 || prof->P < 1 || prof->D < 1 || prof->A < 1 || prof->J < 1 || prof->ROLES < 1 || prof->F < 1 ||
      prof->S > 256 || prof->M > 256 || prof->P > 256 || prof->D > 256 || prof->ROLES > 256)
    return DYPLAN_ERR_LIMIT;
  if (!(prof->token_norm > 0.0f)) return DYPLAN_ERR_ARG;
  ctx->last_launches = 0;
  ctx->have_events = false;
  ctx->last_stream = (cudaStream_t)stream;
  if (NN == 0) return DYPLAN_OK;
  if (!prof->quality || !prof->tokens || !prof->theta_dec || !prof->tau_pre_us || !prof->psi || !opt_off || !pred_mask || !skill ||
      !role || !vuln || (KK > 0 && (!model || !backend || !policy || !acc || !lat_us || !cost)))
    return DYPLAN_ERR_NULL;
  CK(cudaSetDevice(ctx->device));
  BindArgs a;
  memset(&a, 0, sizeof(a));
  a.prof = *prof; a.NN = NN; a.KK = KK; a.opt_off = opt_off; a.pred_mask = pred_mask; a.skill = skill; a.role = role;
  a.model = model; a.backend = backend; a.policy = policy; a.vuln = vuln; a.acc = acc; a.lat_us = lat_us; a.cost = cost;
  a.demand = demand;
  CK(launch_bind(a, (cudaStream_t)stream));
  ctx->last_launches = 1;
  return DYPLAN_OK;
}

int dyplan_compile_linear(dyplan_ctx* ctx, const dyplan_batch* in, const float* cost, const dyplan_linear_params* params, int32_t L,
                          const float* levels, dyplan_bundle* out, const dyplan_linear_extra* extra, void* stream) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = check_batch(in, true);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  cudaStream_t s = (cudaStream_t)stream;
  ctx->last_launches = 0;
  ctx->have_events = false;
  ctx->last_stream = s;
  ctx->last_L = L;
  ctx->last_linear = true;
  if (in->R == 0) return DYPLAN_OK;
  if (!params || !levels || (in->KK > 0 && !cost)) return DYPLAN_ERR_NULL;
  if ((rc = check_bundle(out))) return rc;
  const float pv[6] = {params->lambda_f, params->lambda_c, params->lambda_l, params->lambda_ld, params->beta, params->effort};
  for (float v : pv) if (!(v >= 0.0f) || v > 1e6f) return DYPLAN_ERR_ARG;   // (padding options score -1e30)
  if (params->effort > 1.0f) return DYPLAN_ERR_ARG;
  for (int l = 0; l < L; l++) if (!(levels[l] >= 0.0f) || levels[l] > 1e6f) return DYPLAN_ERR_ARG;
  CK(cudaSetDevice(ctx->device));
  if ((rc = order_after_previous(ctx, s))) return rc;
  const size_t R = (size_t)in->R;
  if ((rc = ensure(ctx, ctx->lin_blob, R * kLinBlobWords * 4))) return rc;
  if ((rc = ensure(ctx, ctx->lin_misc, 64))) return rc;
  LinArgs a;
  memset(&a, 0, sizeof(a));
  a.in = *in; a.out = *out; if (extra) a.extra = *extra; a.cost = cost; a.p = *params; a.L = L;
  for (int l = 0; l < L; l++) a.levels[l] = levels[l];
  a.blob = (uint32_t*)ctx->lin_blob.p;
  a.counter = (uint32_t*)ctx->lin_misc.p; a.plans = (unsigned long long*)((char*)ctx->lin_misc.p + 16);
  const int grid = ctx->sm_count * 8;                         // persistent-ish: work pulled from a device counter
  const uint32_t want = (uint32_t)grid * 4u * 6u;             // ~6 work items per launched warp
  uint32_t chunks = (uint32_t)((want + R - 1) / R);
  a.chunks = chunks < 1 ? 1 : (chunks > 65536u ? 65536u : chunks);
  if ((rc = ensure(ctx, ctx->lin_gj, R * a.chunks * L * sizeof(LinRec)))) return rc;
  a.rec = (LinRec*)ctx->lin_gj.p;
  if ((rc = ensure(ctx, ctx->lin_gkey, R * L * 4))) return rc;
  a.gJ = (int32_t*)ctx->lin_gkey.p;
  CK(cudaMemsetAsync(ctx->lin_misc.p, 0, 64, s));
  CK(cudaEventRecord(ctx->ev0, s));
  CK(launch_linear(a, grid, s));
  CK(cudaEventRecord(ctx->ev1, s));
  ctx->have_events = true;
  ctx->last_launches = 3;
  return mark_done(ctx, s);
}

int dyplan_measure_issue_rates(dyplan_ctx* ctx, dyplan_issue_rate* out, int32_t capacity, int32_t* n_out, float* sm_clock_mhz,
                               void* stream) {
  if (!ctx || !out || !n_out) return DYPLAN_ERR_NULL;
  if (capacity < 1) return DYPLAN_ERR_ARG;
  *n_out = 0;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  const int grid = ctx->sm_count, wpb = m0_warps_per_block();
  const size_t nst = (size_t)grid * wpb * 2;
  int rc;
  if ((rc = ensure(ctx, ctx->arena, nst * sizeof(long long) + 256))) return rc;
  long long* d_st = (long long*)ctx->arena.p;
  float* d_sink = (float*)((char*)ctx->arena.p + nst * sizeof(long long));
  long long* h_st = new (std::nothrow) long long[nst];
  float* rates = new (std::nothrow) float[grid];
  if (!h_st || !rates) { delete[] h_st; delete[] rates; return DYPLAN_ERR_ARG; }
  const int n = m0_count() < capacity ? m0_count() : capacity;
  double clk_sum = 0.0;
  int clk_n = 0;
  cudaError_t e = cudaSuccess;
  for (int op = 0; op < n && e == cudaSuccess; op++) {
    if ((e = m0_launch(op, grid, d_st, d_sink, s)) != cudaSuccess) break;   // warm-up (instruction cache, clocks)
    if ((e = cudaEventRecord(ctx->ev0, s)) != cudaSuccess) break;
    if ((e = m0_launch(op, grid, d_st, d_sink, s)) != cudaSuccess) break;
    if ((e = cudaEventRecord(ctx->ev1, s)) != cudaSuccess) break;
    if ((e = cudaMemcpyAsync(h_st, d_st, nst * sizeof(long long), cudaMemcpyDeviceToHost, s)) != cudaSuccess) break;
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) break;
    float ms = 0.f;
    if ((e = cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1)) != cudaSuccess) break;
    long long longest = 0;
    for (int b = 0; b < grid; b++) {
      long long t0 = h_st[(size_t)b * wpb * 2], t1 = h_st[(size_t)b * wpb * 2 + 1];
      for (int w = 1; w < wpb; w++) {
        const long long a0 = h_st[((size_t)b * wpb + w) * 2], a1 = h_st[((size_t)b * wpb + w) * 2 + 1];
        t0 = a0 < t0 ? a0 : t0; t1 = a1 > t1 ? a1 : t1;
      }
      const long long cyc = t1 - t0 > 0 ? t1 - t0 : 1;
      longest = cyc > longest ? cyc : longest;
      rates[b] = (float)((double)wpb * m0_warp_inst_per_warp() / 4.0 / (double)cyc);
    }
    for (int i = 1; i < grid; i++) {   // insertion sort: grid = 148
      const float v = rates[i]; int j = i - 1;
      while (j >= 0 && rates[j] > v) { rates[j + 1] = rates[j]; j--; }
      rates[j + 1] = v;
    }
    memset(out[op].name, 0, sizeof(out[op].name));
    strncpy(out[op].name, m0_name(op), sizeof(out[op].name) - 1);
    out[op].rate = rates[grid / 2]; out[op].rate_min = rates[0]; out[op].rate_max = rates[grid - 1];
    if (ms > 0.f) { clk_sum += (double)longest / ((double)ms * 1e3); clk_n++; }   // cycles per microsecond = MHz
  }
  delete[] h_st; delete[] rates;
  if (e != cudaSuccess) return fail_cuda(ctx, e);
  *n_out = n;
  if (sm_clock_mhz) *sm_clock_mhz = clk_n ? (float)(clk_sum / clk_n) : 0.f;
  ctx->last_launches = 2 * n; ctx->have_events = false; ctx->last_stream = s;
  return DYPLAN_OK;
}

int dyplan_last_stats(dyplan_ctx* ctx, dyplan_stats* out) {
  if (!ctx || !out) return DYPLAN_ERR_NULL;
  memset(out, 0, sizeof(*out));
  out->sm_count = ctx->sm_count;
  out->launches = ctx->last_launches;
  CK(cudaSetDevice(ctx->device));
  CK(cudaStreamSynchronize(ctx->last_stream));
  if (ctx->have_events && ctx->last_linear && ctx->lin_misc.p) {
    unsigned long long plans = 0;
    CK(cudaMemcpy(&plans, (char*)ctx->lin_misc.p + 16, 8, cudaMemcpyDeviceToHost));
    out->plans = plans;
    out->evals = plans * (uint64_t)ctx->last_L;
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    out->score_ms = ms;
  } else if (ctx->have_events && ctx->state.p) {
    CallState st;
    CK(cudaMemcpy(&st, ctx->state.p, sizeof(st), cudaMemcpyDeviceToHost));
    out->plans = st.total_plans;
    out->evals = st.total_plans * (uint64_t)ctx->last_L;
    out->work_items = (uint64_t)st.total_items + st.total_items_f;
    out->fast_requests = st.fast_requests;
    out->slow_steps = st.slow_steps;
    out->bound_skipped = st.bound_skipped;
    out->approx_requests = st.approx_requests;
    out->small_requests = st.small_requests;
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    out->score_ms = ms;
  }
  return DYPLAN_OK;
}

}  // extern "C"

// ---- *_host calls: stage the copies, run the same kernels, copy back ---------------------------------------------
namespace {

struct Arena {
  char* base;
  size_t off;
  char* stage = nullptr;   // pinned host image (small calls), else null
  template <typename T>
  T* take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    T* p = (T*)(base + off);
    off += n * sizeof(T);
    return p;
  }
};

struct HostPlan {   // sizes of everything a call moves
  size_t R, NN, KK, B, L, nrec;
};

size_t arena_bytes(const HostPlan& p) {
  // generous: every array rounded to 256 B
  size_t n = 0;
  auto add = [&](size_t bytes) { n += ((bytes + 255) & ~(size_t)255) + 256; };
  add((p.R + 1) * 4); add((p.NN + 1) * 4); add(p.NN * 4); add(p.NN * 4);
  add(p.KK * 4); add(p.KK * 4); add(p.KK * 4); add(p.KK); add(p.KK);
  add(p.R * 4); add(p.R * p.B * 4);
  add(p.L * p.B * 4 + p.R * p.B * 4); add(p.R * 4); add(p.NN);
  // outputs (two bundles at most: stored + rescored) + variant
  for (int i = 0; i < 2; i++) {
    add(p.nrec * 8); add(p.nrec * 16); add(p.nrec * 4); add(p.nrec * 8); add(p.nrec * 4); add(p.nrec * p.B * 4); add(p.nrec); add(p.nrec);
  }
  add(p.R * 4);
  add(p.KK * 4); add(p.nrec * 4); add(p.nrec * 8);   // linear mode: cost, dtau, quality
  return n;
}

}  // namespace

// A small call is dominated by the fixed cost of its copies (12-14 cudaMemcpyAsync in, 8 out): below kStageBytes the
// inputs are packed into a pinned image of the arena and travel as ONE copy each way; larger calls copy each array
// straight from the caller's buffer (packing 27 MB on the host would cost more than it saves).
constexpr size_t kStageBytes = 256 << 10;
constexpr size_t kZeroCopyBytes = 8 << 10;   // input images up to this size are fetched by k_stage itself (no DMA copies)
#define H2D(dst, src, n, T)                                                                            \
  do {                                                                                                 \
    dst = ar.take<T>(n);                                                                               \
    if ((n) > 0) {                                                                                     \
      if (ar.stage) memcpy(ar.stage + ((char*)dst - ar.base), src, (size_t)(n) * sizeof(T));           \
      else CK(cudaMemcpyAsync((void*)dst, src, (size_t)(n) * sizeof(T), cudaMemcpyHostToDevice, s));   \
      h2d += (size_t)(n) * sizeof(T);                                                                  \
    }                                                                                                  \
  } while (0)

static int batch_to_device(dyplan_ctx* ctx, const dyplan_batch* in, Arena& ar, dyplan_batch* d, cudaStream_t s, uint64_t& h2d) {
  *d = *in;
  int32_t *node_off, *opt_off, *lat, *dem, *slo, *cap = nullptr;
  uint32_t* pm; float *vuln, *acc; uint8_t *be, *mo;
  H2D(node_off, in->node_off, (size_t)in->R + 1, int32_t);
  H2D(opt_off, in->opt_off, (size_t)in->NN + 1, int32_t);
  H2D(pm, in->pred_mask, (size_t)in->NN, uint32_t);
  H2D(vuln, in->vuln, (size_t)in->NN, float);
  H2D(lat, in->lat_us, (size_t)in->KK, int32_t);
  H2D(acc, in->acc, (size_t)in->KK, float);
  H2D(dem, in->demand, (size_t)in->KK, int32_t);
  H2D(be, in->backend, (size_t)in->KK, uint8_t);
  H2D(mo, in->model, (size_t)in->KK, uint8_t);
  H2D(slo, in->slo_us, (size_t)in->R, int32_t);
  if (in->cap) H2D(cap, in->cap, (size_t)in->R * in->B, int32_t);
  d->node_off = node_off; d->opt_off = opt_off; d->pred_mask = pm; d->vuln = vuln; d->lat_us = lat; d->acc = acc;
  d->demand = dem; d->backend = be; d->model = mo; d->slo_us = slo; d->cap = cap;
  return DYPLAN_OK;
}

static void bundle_alloc(Arena& ar, size_t nrec, size_t B, bool want64, dyplan_bundle* d) {
  d->plan_idx = ar.take<uint64_t>(nrec); d->choice = ar.take<uint8_t>(nrec * 16); d->corr = ar.take<float>(nrec);
  d->corr64 = want64 ? ar.take<double>(nrec) : nullptr; d->lat = ar.take<int32_t>(nrec); d->dem = ar.take<int32_t>(nrec * B);
  d->dom_model = ar.take<uint8_t>(nrec); d->status = ar.take<uint8_t>(nrec);
}

#define D2H(dst, src, n, T)                                                                              \
  do {                                                                                                   \
    if ((n) > 0 && (dst)) {                                                                              \
      if (stage) memcpy((void*)(dst), stage + ((const char*)(src) - abase), (size_t)(n) * sizeof(T));    \
      else CK(cudaMemcpyAsync((void*)(dst), src, (size_t)(n) * sizeof(T), cudaMemcpyDeviceToHost, s));   \
      d2h += (size_t)(n) * sizeof(T);                                                                    \
    }                                                                                                    \
  } while (0)

// stage != null: the device arena's output region is already in the pinned image (one copy, synchronised): scatter it
static int bundle_to_host(dyplan_ctx* ctx, const dyplan_bundle* d, dyplan_bundle* h, size_t nrec, size_t B, cudaStream_t s, uint64_t& d2h,
                          const char* stage = nullptr, const char* abase = nullptr) {
  D2H(h->plan_idx, d->plan_idx, nrec, uint64_t);
  D2H(h->choice, d->choice, nrec * 16, uint8_t);
  D2H(h->corr, d->corr, nrec, float);
  if (d->corr64) D2H(h->corr64, d->corr64, nrec, double);
  D2H(h->lat, d->lat, nrec, int32_t);
  D2H(h->dem, d->dem, nrec * B, int32_t);
  D2H(h->dom_model, d->dom_model, nrec, uint8_t);
  D2H(h->status, d->status, nrec, uint8_t);
  return DYPLAN_OK;
}

static int host_sizes_ok(const dyplan_batch* in) {
  int rc = check_batch(in, true);
  if (rc) return rc;
  if (in->R > 0 && (in->node_off[in->R] != in->NN)) return DYPLAN_ERR_ARG;
  if (in->R > 0 && in->NN > 0 && in->opt_off[in->NN] != in->KK) return DYPLAN_ERR_ARG;
  return DYPLAN_OK;
}

static int solve_host(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult, const uint32_t* dispatched,
                      const uint8_t* fixed_choice, uint32_t flags, bool is_replan, dyplan_bundle* out, void* stream,
                      uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = host_sizes_ok(in);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  uint64_t h2d = 0, d2h = 0;
  if (h2d_bytes) *h2d_bytes = 0;
  if (d2h_bytes) *d2h_bytes = 0;
  if (in->R == 0) return DYPLAN_OK;
  if (!mult || (is_replan && (!dispatched || (in->NN > 0 && !fixed_choice)))) return DYPLAN_ERR_NULL;
  if ((rc = check_bundle(out))) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  HostPlan hp{(size_t)in->R, (size_t)in->NN, (size_t)in->KK, (size_t)in->B, (size_t)L, (size_t)in->R * L};
  const size_t abytes = arena_bytes(hp);
  if ((rc = ensure(ctx, ctx->arena, abytes))) return rc;
  Arena ar{(char*)ctx->arena.p, 0};
  if (abytes <= kStageBytes) {
    if (ctx->hstage_cap < kStageBytes) {
      if (ctx->hstage) CK(cudaFreeHost(ctx->hstage));
      ctx->hstage = nullptr; ctx->hstage_cap = 0;
      CK(cudaHostAlloc(&ctx->hstage, kStageBytes, cudaHostAllocDefault));
      ctx->hstage_cap = kStageBytes;
    }
    ar.stage = (char*)ctx->hstage;
  }
  dyplan_batch d;
  if ((rc = batch_to_device(ctx, in, ar, &d, s, h2d))) return rc;
  int32_t* dmult; uint32_t* ddisp = nullptr; uint8_t* dfix = nullptr;
  H2D(dmult, mult, is_replan ? (size_t)in->R * in->B : (size_t)L * in->B, int32_t);
  if (is_replan) { H2D(ddisp, dispatched, (size_t)in->R, uint32_t); H2D(dfix, fixed_choice, (size_t)in->NN, uint8_t); }
  // A tiny call (one admission-time compile is a few hundred bytes in, a few hundred out) does not use the copy engine at
  // all: k_stage fetches the image from the pinned buffer itself and the kernels store the records straight into it
  // (pinned memory is device-visible at the same address); what is left of the call is two launches and a synchronise.
  const size_t in_bytes = ar.off;
  const bool zero_copy = ar.stage && in_bytes <= kZeroCopyBytes;
  if (ar.stage && !zero_copy) CK(cudaMemcpyAsync(ar.base, ar.stage, ar.off, cudaMemcpyHostToDevice, s));   // the whole input image, once
  const size_t out_begin = (ar.off + 255) & ~(size_t)255;
  dyplan_bundle dout;
  bundle_alloc(ar, hp.nrec, hp.B, out->corr64 != nullptr, &dout);
  if (zero_copy) {   // the records' home is the pinned image
    const ptrdiff_t sh = ar.stage - ar.base;
    dout.plan_idx = (uint64_t*)((char*)dout.plan_idx + sh); dout.choice = (uint8_t*)((char*)dout.choice + sh);
    dout.corr = (float*)((char*)dout.corr + sh); if (dout.corr64) dout.corr64 = (double*)((char*)dout.corr64 + sh);
    dout.lat = (int32_t*)((char*)dout.lat + sh); dout.dem = (int32_t*)((char*)dout.dem + sh);
    dout.dom_model = (uint8_t*)((char*)dout.dom_model + sh); dout.status = (uint8_t*)((char*)dout.status + sh);
  }
  // every request small enough for k_small (an upper bound of what k_stage will find: pinned nodes only shrink it)?
  bool all_small = in->R <= kSmallMaxR;
  for (int32_t r = 0; r < in->R && all_small; r++) {
    const int32_t n0 = in->node_off[r], n1 = in->node_off[r + 1];
    if (n0 < 0 || n1 < n0 || n1 > in->NN) break;   // malformed: k_stage reports it
    unsigned long long p = 1;
    for (int32_t n = n0; n < n1 && all_small; n++) {
      const long long k = (long long)in->opt_off[n + 1] - in->opt_off[n];
      if (k >= 1 && k <= DYPLAN_MAX_OPTS) p *= (unsigned long long)k;
      if (p * (unsigned long long)L > kSmallMaxEvals) all_small = false;
    }
  }
  if ((rc = run_solve(ctx, &d, L, dmult, ddisp, dfix, flags, is_replan, &dout, s, all_small, zero_copy ? ar.stage : nullptr,
                      zero_copy ? ar.base : nullptr, zero_copy ? in_bytes : 0))) return rc;
  if (zero_copy) {
    CK(cudaStreamSynchronize(s));
    if ((rc = bundle_to_host(ctx, &dout, out, hp.nrec, hp.B, s, d2h, ar.stage, ar.stage))) return rc;
  } else if (ar.stage) {
    CK(cudaMemcpyAsync(ar.stage + out_begin, ar.base + out_begin, ar.off - out_begin, cudaMemcpyDeviceToHost, s));   // every record, once
    CK(cudaStreamSynchronize(s));
    if ((rc = bundle_to_host(ctx, &dout, out, hp.nrec, hp.B, s, d2h, ar.stage, ar.base))) return rc;
  } else {
    if ((rc = bundle_to_host(ctx, &dout, out, hp.nrec, hp.B, s, d2h))) return rc;
    CK(cudaStreamSynchronize(s));
  }
  if (h2d_bytes) *h2d_bytes = h2d;
  if (d2h_bytes) *d2h_bytes = d2h;
  return DYPLAN_OK;
}

extern "C" {

int dyplan_compile_host(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult_pm, dyplan_bundle* out,
                        void* stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  return solve_host(ctx, in, L, mult_pm, nullptr, nullptr, 0, false, out, stream, h2d_bytes, d2h_bytes);
}

int dyplan_replan_host(dyplan_ctx* ctx, const dyplan_batch* in, const uint32_t* dispatched_mask, const uint8_t* fixed_choice,
                       const int32_t* live_mult_pm, uint32_t flags, dyplan_bundle* out, void* stream, uint64_t* h2d_bytes,
                       uint64_t* d2h_bytes) {
  if (flags & ~DYPLAN_RESIDUAL) return DYPLAN_ERR_ARG;
  return solve_host(ctx, in, 1, live_mult_pm, dispatched_mask, fixed_choice, flags, true, out, stream, h2d_bytes, d2h_bytes);
}

int dyplan_compile_linear_host(dyplan_ctx* ctx, const dyplan_batch* in, const float* cost, const dyplan_linear_params* params, int32_t L,
                               const float* levels, dyplan_bundle* out, const dyplan_linear_extra* extra, void* stream,
                               uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = host_sizes_ok(in);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  uint64_t h2d = 0, d2h = 0;
  if (h2d_bytes) *h2d_bytes = 0;
  if (d2h_bytes) *d2h_bytes = 0;
  if (in->R == 0) return DYPLAN_OK;
  if (!params || !levels || (in->KK > 0 && !cost)) return DYPLAN_ERR_NULL;
  if ((rc = check_bundle(out))) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  HostPlan hp{(size_t)in->R, (size_t)in->NN, (size_t)in->KK, (size_t)in->B, (size_t)L, (size_t)in->R * L};
  if ((rc = ensure(ctx, ctx->arena, arena_bytes(hp)))) return rc;
  Arena ar{(char*)ctx->arena.p, 0};
  dyplan_batch d;
  if ((rc = batch_to_device(ctx, in, ar, &d, s, h2d))) return rc;
  float* dcost;
  H2D(dcost, cost, (size_t)in->KK, float);
  dyplan_bundle dout;
  bundle_alloc(ar, hp.nrec, hp.B, out->corr64 != nullptr, &dout);
  dyplan_linear_extra dex;
  dex.dtau = (extra && extra->dtau) ? ar.take<int32_t>(hp.nrec) : nullptr;
  dex.quality = (extra && extra->quality) ? ar.take<double>(hp.nrec) : nullptr;
  const char* stage = nullptr; const char* abase = nullptr;   // (this entry point copies array by array)
  if ((rc = dyplan_compile_linear(ctx, &d, dcost, params, L, levels, &dout, &dex, stream))) return rc;
  if ((rc = bundle_to_host(ctx, &dout, out, hp.nrec, hp.B, s, d2h))) return rc;
  if (dex.dtau) D2H(extra->dtau, dex.dtau, hp.nrec, int32_t);
  if (dex.quality) D2H(extra->quality, dex.quality, hp.nrec, double);
  CK(cudaStreamSynchronize(s));
  if (h2d_bytes) *h2d_bytes = h2d;
  if (d2h_bytes) *d2h_bytes = d2h;
  return DYPLAN_OK;
}

int dyplan_select_host(dyplan_ctx* ctx, const dyplan_batch* in, const dyplan_bundle* bundle, int32_t L, const int32_t* live_mult_pm,
                       int32_t* variant, dyplan_bundle* rescored, void* stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  if (!ctx) return DYPLAN_ERR_NULL;
  int rc = host_sizes_ok(in);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  uint64_t h2d = 0, d2h = 0;
  if (h2d_bytes) *h2d_bytes = 0;
  if (d2h_bytes) *d2h_bytes = 0;
  if (in->R == 0) return DYPLAN_OK;
  if (!bundle || !bundle->choice || !bundle->status || !live_mult_pm || !variant) return DYPLAN_ERR_NULL;
  if (rescored && (rc = check_bundle(rescored))) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaSetDevice(ctx->device));
  HostPlan hp{(size_t)in->R, (size_t)in->NN, (size_t)in->KK, (size_t)in->B, (size_t)L, (size_t)in->R * L};
  if ((rc = ensure(ctx, ctx->arena, arena_bytes(hp)))) return rc;
  Arena ar{(char*)ctx->arena.p, 0};
  dyplan_batch d;
  if ((rc = batch_to_device(ctx, in, ar, &d, s, h2d))) return rc;
  int32_t* dlive; uint8_t *dch, *dst;
  H2D(dlive, live_mult_pm, (size_t)in->B, int32_t);
  H2D(dch, bundle->choice, hp.nrec * 16, uint8_t);
  H2D(dst, bundle->status, hp.nrec, uint8_t);
  dyplan_bundle dbundle;
  memset(&dbundle, 0, sizeof(dbundle));
  dbundle.choice = dch; dbundle.status = dst;
  int32_t* dvar = ar.take<int32_t>(hp.R);
  dyplan_bundle dres;
  if (rescored) bundle_alloc(ar, hp.R, hp.B, rescored->corr64 != nullptr, &dres);
  const char* stage = nullptr; const char* abase = nullptr;   // (this entry point copies array by array)
  if ((rc = dyplan_select(ctx, &d, &dbundle, L, dlive, dvar, rescored ? &dres : nullptr, stream))) return rc;
  D2H(variant, dvar, hp.R, int32_t);
  if (rescored && (rc = bundle_to_host(ctx, &dres, rescored, hp.R, hp.B, s, d2h))) return rc;
  CK(cudaStreamSynchronize(s));
  if (h2d_bytes) *h2d_bytes = h2d;
  if (d2h_bytes) *d2h_bytes = d2h;
  return DYPLAN_OK;
}

}  // extern "C"

// ---- dyplan_compile_static: the compile call with no device allocation (include/dyplan.h) -------------------------
// The scorers' scratch normally lives in buffers the ctx grows with cudaMalloc.  Here it is carved from one file-scope
// device array, so the call is usable where cudaMalloc is not (graph capture, serving loops).  The array is shared by
// every ctx and call on a device and keeps the last call's contents: k_stage / k_plan reset the tickets, thresholds and
// counters at the start of every call, exactly as they do for the ctx's own (equally unzeroed, reused) buffers.
static __device__ __align__(256) unsigned char g_static_scratch[DYPLAN_STATIC_SCRATCH_BYTES];

namespace {

// In host code `g_static_scratch` is only the host-side shadow of the symbol, not a device address: the address the
// kernels can use is looked up once per device, with that device current, and cached.
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
unsigned char* g_static_ptr[kStaticMaxDevices];   // zero-initialised: not looked up yet

cudaError_t static_scratch_base(int device, unsigned char** base) {
  if (device < 0 || device >= kStaticMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);   // the caller made `device` current
    if (e != cudaSuccess) return e;
    if (!p || ((uintptr_t)p & 255u)) return cudaErrorInvalidSymbol;
    g_static_ptr[device] = (unsigned char*)p;
  }
  *base = g_static_ptr[device];
  return cudaSuccess;
}

struct StaticCarver {   // 256-byte aligned pieces of the array; `off` is what the layout needs in total
  unsigned char* base;
  size_t off = 0;
  template <typename T>
  T* take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    T* p = (T*)(base + off);
    off += n * sizeof(T);
    return p;
  }
};

// work-item budget of a static call: 2R+2 records of rounding slack plus 32768 items per scorer class (k_plan cuts
// coarser items when a class would need more, so any plan space still fits)
constexpr uint32_t kStaticItemsPerClass = 32768;

}  // namespace

extern "C" int dyplan_compile_static(dyplan_ctx* ctx, const dyplan_batch* in, int32_t L, const int32_t* mult_pm, dyplan_bundle* out,
                                     void* stream_) {
  if (!ctx) return DYPLAN_ERR_NULL;
  cudaStream_t stream = (cudaStream_t)stream_;
  int rc = check_batch(in, true);
  if (rc) return rc;
  if (L < 1 || L > DYPLAN_MAX_LEVELS) return DYPLAN_ERR_LIMIT;
  ctx->last_launches = 0;
  ctx->have_events = false;   // (dyplan_last_stats: launches and sm_count only)
  ctx->last_stream = stream;
  ctx->last_L = L;
  ctx->last_linear = false;
  if (in->R == 0) return DYPLAN_OK;
  if (!mult_pm) return DYPLAN_ERR_NULL;
  if ((rc = check_bundle(out))) return rc;
  if (in->R > DYPLAN_STATIC_MAX_REQUESTS) {
    snprintf(ctx->errbuf, sizeof(ctx->errbuf), "dyplan_compile_static: R = %d requests exceed DYPLAN_STATIC_MAX_REQUESTS = %d "
             "(static scratch of %u bytes); use dyplan_compile", (int)in->R, DYPLAN_STATIC_MAX_REQUESTS, (unsigned)DYPLAN_STATIC_SCRATCH_BYTES);
    return DYPLAN_ERR_STATIC_LIMIT;
  }
  CK(cudaSetDevice(ctx->device));
  unsigned char* base = nullptr;
  CK(static_scratch_base(ctx->device, &base));

  const size_t R = (size_t)in->R;
  const int nbc = nb_class_of(in->B, in->cap != nullptr);
  int& occ = ctx->occ[L - 1][nb_index(nbc)];
  if (occ <= 0) {
    occ = kOcc[L - 1](nbc);
    if (occ <= 0) return fail_cuda(ctx, cudaGetLastError() == cudaSuccess ? cudaErrorLaunchOutOfResources : cudaPeekAtLastError());
  }
  int& focc = ctx->focc[L - 1];
  if (focc <= 0) {
    focc = kFOcc[L - 1]();
    if (focc <= 0) return fail_cuda(ctx, cudaGetLastError() == cudaSuccess ? cudaErrorLaunchOutOfResources : cudaPeekAtLastError());
  }
  const int grid = ctx->sm_count * occ;
  const int fgrid = ctx->sm_count * focc;
  const uint32_t target_items_f = (uint32_t)(fgrid * kFastWarps) * fast_items_per_warp(focc);
  const uint32_t max_items = (uint32_t)(2 * R + 2) + 2u * kStaticItemsPerClass;

  CallArgs a;
  memset(&a, 0, sizeof(a));
  a.in = *in; a.out = *out; a.L = L; a.mult = mult_pm; a.ctx_flags = ctx->flags;
  a.small_mode = (in->R <= kSmallMaxR && !(ctx->flags & DYPLAN_NO_SMALL_PATH)) ? 1 : 0;
  a.small_split = a.small_mode ? (kSmallBlocksPerSm * ctx->sm_count / (int)in->R > 1 ? kSmallBlocksPerSm * ctx->sm_count / (int)in->R : 1) : 1;
  StaticCarver sc{base};
  a.blob = sc.take<uint32_t>(R * blob_stride_words(L));
  a.item_off = sc.take<uint32_t>(2 * (R + 1)); a.item_off_f = a.item_off + (R + 1);
  a.done = sc.take<uint32_t>(R);
  a.gthr = sc.take<float>(R * L);
  // k_small writes small_split records per request, the batched scorers one per work item: room for the larger
  const size_t small_recs = a.small_mode ? R * (size_t)a.small_split : 0;
  a.partial = sc.take<Partial>((small_recs > max_items ? small_recs : (size_t)max_items) * L);
  a.st = sc.take<CallState>(1);
  a.target_items_f = target_items_f; a.fast_warps = (uint32_t)(fgrid * kFastWarps);
  a.max_items = max_items;
  if (sc.off > (size_t)DYPLAN_STATIC_SCRATCH_BYTES) {   // (cannot happen within the limits above: a guard for a device with > 1000 SMs)
    snprintf(ctx->errbuf, sizeof(ctx->errbuf), "dyplan_compile_static: the scratch layout needs %zu bytes, the static array holds %u",
             sc.off, (unsigned)DYPLAN_STATIC_SCRATCH_BYTES);
    return DYPLAN_ERR_STATIC_LIMIT;
  }

  CK(launch_stage(a, stream));
  int launches = 1;
  if (a.small_mode) { CK(launch_small(a, stream)); launches++; }
  if (!(a.small_mode && sizes_prove_all_small(in, L))) {
    CK(launch_seed(a, stream));
    CK(launch_plan(a, stream));
    CK(kFLaunch[L - 1](a, fgrid, stream));
    CK(kLaunch[L - 1](a, nbc, grid, stream));
    launches += 4;
  }
  ctx->last_launches = launches;
  return DYPLAN_OK;
}
