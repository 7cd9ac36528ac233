// dyplan_internal.cuh -- structures shared by the kernels of libdyplan (product side only; the oracle
// shares nothing with this directory).  See DESIGN.md sections 6-7 for the layout and the kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dyplan.h"

namespace dyplan {

constexpr int kBlock = 128;          // threads per scoring block
constexpr int kMinBlocks = 4;        // resident scoring blocks per SM the register allocation is bounded for
constexpr int kHdrWords = 124;       // ReqHdr size in 4-byte words (multiple of 4 -> 16-byte aligned tables)
constexpr int kMaxSlots = 16 * 16 + 4;  // option slots of one request incl. dummies, padded to 4
constexpr int kDem0bWords = 16 * 8;  // per-backend demand of the inner node's options [k0][b]
constexpr int kMaxBlobWords = kHdrWords + kDem0bWords + kMaxSlots * (DYPLAN_MAX_LEVELS + 3);
// Every request owns a fixed-size blob (header, dem0b, lat[slot][L], f[slot], dem[slot], be[slot]); only the used
// part is ever written or read, so the stride costs address space, not traffic.
__host__ __device__ inline size_t blob_stride_words(int L) { return (size_t)kHdrWords + kDem0bWords + (size_t)kMaxSlots * (size_t)(L + 3); }
constexpr uint64_t kNoIdx = ~0ull;
constexpr int kClassWide = 0;        // int32 slack DP (k_score): any request the ABI admits
constexpr int kClassFast = 1;        // fp32 slack DP (k_fscore): exact when every latency / demand sum is below 2^22, else a
                                     // conservative screen whose candidates are verified in int32 (ReqHdr.approx); tables <= kFastBlobWords
constexpr int kClassSmall = 2;       // a small request of a small call: int32 layout, solved by k_small (dyplan_small.cu)
constexpr int kSmallMaxR = 32;       // calls of at most this many requests try the small path
constexpr int kSmallThreads = 128;
constexpr int kSmallBlocksPerSm = 4;   // blocks of k_small per SM that the requests of a call share (2, 3, 4, 6, 8, 12 measured on configs[0]: 70 / 64 / 60 / 62 / 65 / 67 us)
constexpr unsigned long long kSmallMaxEvals = 1ull << 21;   // (plan, level) evaluations of a request k_small takes
constexpr int kFastBlobWords = 1536; // per-warp shared-memory window of k_fscore (6 KB)
constexpr int kFastWarps = 4;        // warps per k_fscore block (each warp works on its own item)
// work items to aim for per resident warp of k_fscore.  Measured on configs[1..4] (kernel ms): with 4 blocks per SM
// (L <= 4) 8 / 10 / 12 / 16 items give 2.555 / 2.532 / 2.566 / 2.699 on configs[1]; with 3 blocks per SM (L >= 6)
// 8 / 10 / 12 / 16 / 24 give 52.0 / 49.4 / 48.8 / 49.6 / 51.0 on configs[4]: about 36-40 items per scheduler either way
// (fewer: a longer tail; more: the per-item prologue, ticket and fence)
__host__ __device__ inline uint32_t fast_items_per_warp(int blocks_per_sm) { return blocks_per_sm >= 4 ? 10u : 12u; }
constexpr float kBigF = 1099511627776.0f; // 2^40: above every slack, latency and demand the ABI admits (< 2^31)
// fast class: outer indices per work item of a request whose node 2 has K2 options -- the call-wide figure rounded up
// so that each of the 32 lanes gets a whole number of node-2 sweeps (no idle-lane tail inside full items)
__host__ __device__ inline unsigned long long fast_item_outer(unsigned long long pif, int K2, bool small_call) {
  const unsigned long long q = 32ull * (unsigned long long)(K2 < 1 ? 1 : K2);
  if (small_call) return ((pif + 31) / 32) * 32;   // too little work to fill the GPU: favour more items over aligned lanes
  return ((pif + q - 1) / q) * q;
}
__host__ __device__ inline int level_class(int L) { return L <= 4 ? L : (L <= 6 ? 6 : 8); }

// Per-request staged problem in "internal" node order.  Internal node 0 is the innermost
// enumeration digit, node 1 the middle digit, nodes >= 2 the outer digits.  deps(i) only holds nodes j > i, so
// the slack recurrence  u[i] = min(SLO, min_{j in deps(i)} u[j]) - d[i][k_i]  can be evaluated from the
// outermost node inwards; the longest path is  T = SLO - min_i u[i]  (Eq.(3), in slack form).
struct ReqHdr {
  int32_t status;        // DYPLAN_ST_OK, _INVALID or _TOO_LARGE (input problems only)
  int32_t n_int;         // internal nodes N' >= 3 (dummy nodes appended when N < 3)
  int32_t n_orig;        // original nodes N
  int32_t orient;        // 0: internal i = original i, deps = successors; 1: internal i = original N-1-i, deps = predecessors
  int32_t K0, K1;        // real radices of internal nodes 0 and 1
  int32_t K0p;           // inner radix class: K0 padded up to one of {2,4,6,8,12,16}
  int32_t slo;
  int32_t nslots_pad;    // option slots in the tables (multiple of 4)
  int32_t n0;            // first original node (node_off[r])
  int32_t conn01;        // 1 if internal node 1 is in deps(0)
  uint32_t skip_mask;    // original nodes that contribute nothing (RESIDUAL replan)
  unsigned long long outer_total;  // prod_{i>=2} K'_i : number of outer indices
  unsigned long long base_idx;     // canonical-index contribution of the pinned (dispatched) nodes
  int32_t cap[8];        // per-backend caps (INT32_MAX when absent)
  int32_t Kp[16];        // enumerated radix per internal node (1 for pinned / dummy nodes)
  uint32_t deps[16];     // dependency mask per internal node (internal indices, all > i)
  int32_t optbase[16];   // first table slot of internal node i
  // --- fields of the float ("fast") scorer; zero for requests of the wide class ---
  int32_t klass;         // kClassWide or kClassFast
  int32_t nbc;           // cap class of the fast scorer: 0 (no caps) or 2/3/4/8 backend groups of node 0's slots
  int32_t Lp;            // level count padded to the scorer's template class (1,2,3,4,6,8)
  float slo_f;           // min(SLO, longest possible T): every slack is an exact fp32 integer
  float S01;             // 1 if internal node 1 is in deps(0), else 2^24 (turns "u1 >= 0" into a bound that never binds)
  float big12, big02;    // 0 if internal node 2 is in deps(1) / deps(0), else 2^24
  int32_t blob_words;    // words of this request's staged blob (header + tables)
  float capf[8];         // min(cap, largest possible demand) per backend (+big when absent), rounded up
  unsigned long long stride[16];   // canonical stride of internal node i (0 for dummies / pinned nodes)
  int32_t approx;        // 1: a latency or demand sum can exceed 2^22, so the fp32 slacks are upper bounds (directed
                         //    rounding) and every candidate is verified with the int32 tables that follow the fp32 ones
  int32_t slo_c;         // min(SLO, longest possible T) as an integer
  int32_t ioff;          // word offset of the int32 tables ilat[slot][Lp], idem[slot] in the request's blob in GLOBAL memory
                         // (approx only; they follow the blob_words the scorer stages in shared memory)
  int32_t pad1;
};
static_assert(sizeof(ReqHdr) == kHdrWords * 4, "ReqHdr layout");

// partial best of one work item and one level
struct __align__(16) Partial {
  float C;
  int32_t T;
  unsigned long long idx;   // kNoIdx: none
};

// device-side counters / plan of one call
struct CallState {
  unsigned long long total_outer;   // sum over valid requests of outer_total
  unsigned long long total_plans;   // sum over valid requests of enumerated plans
  unsigned long long per_item_outer;   // wide class: outer indices per (block) work item
  unsigned long long per_item_outer_f; // fast class: outer indices per (warp) work item
  unsigned long long slow_steps;
  unsigned long long bound_skipped;    // outer indices the subtree bound skipped (DYPLAN_PRUNE_BOUNDS)
  uint32_t total_items;             // wide class
  uint32_t next_item;               // wide class: dynamic work counter
  uint32_t total_items_f;           // fast class
  uint32_t next_item_f;
  uint32_t fast_requests;           // requests staged for the fp32 scorer
  uint32_t small_call_f;            // fast class: fewer than ~1K outer indices per resident warp (items are not lane-aligned)
  uint32_t tail_start_f;            // fast class: requests >= this index are cut into 4x smaller items (they are handed out last: a short tail)
  uint32_t approx_requests;         // fast class: requests verified in int32 (ReqHdr.approx)
  uint32_t small_requests;          // requests solved by k_small
  uint32_t pad0;
  // fast class: the order in which work items are handed out.  Items are numbered request by request; the t-th item
  // handed out is item (t * perm_sA) mod perm_nA among the first perm_nA (the regular items), then the same with perm_sB
  // among the rest (the small items of the tail); the strides are coprime to the counts and a little above the items of
  // one request, so consecutive hand-outs fall on consecutive requests and every request is visited all along the launch
  uint32_t perm_nA, perm_sA, perm_sB;
  uint32_t perm_sW;                 // wide class: the t-th item handed out is item (t * perm_sW) mod total_items
};
// outer indices per item of request r before rounding (k_plan and k_fscore must agree)
__host__ __device__ inline unsigned long long fast_pif_of(unsigned long long pif, uint32_t tail_start, long long r) {
  return (unsigned long long)r >= tail_start ? (pif / 4 < 32 ? 32 : pif / 4) : pif;
}

struct CallArgs {                   // passed by value to the kernels
  dyplan_batch in;
  dyplan_bundle out;
  int32_t L;
  const int32_t* mult;              // [L*B] (compile) or [R*B] (replan)
  const uint32_t* dispatched;       // replan only
  const uint8_t* fixed_choice;      // replan only
  uint32_t flags;
  uint32_t ctx_flags;               // DYPLAN_PRUNE_DOMINATED | DYPLAN_PRUNE_BOUNDS (dyplan_set_flags)
  int32_t is_replan;
  const uint4* img_src;             // tiny *_host calls: the packed input image in pinned host memory (device-visible), or null
  uint4* img_dst;                   //   ... and where k_stage copies it in the device arena (the batch pointers point there)
  uint32_t img_vec;                 //   ... its length in 16-byte words
  int32_t small_mode;               // R <= kSmallMaxR: requests of at most kSmallMaxEvals evaluations are staged for k_small
  int32_t small_split;              // blocks per request in k_small (about 4 blocks per SM over the call)
  // scratch
  uint32_t* blob;                   // staged requests
  uint32_t* item_off;               // [R+1] wide class
  uint32_t* item_off_f;             // [R+1] fast class (partial records of fast items follow the wide ones)
  uint32_t* done;                   // [R] ticket counters
  float* gthr;                      // [R*L] published best C per (request, level)
  Partial* partial;                 // [max_items * L]
  CallState* st;
  uint32_t max_items;               // bound on wide items + fast items
  uint32_t target_items_f;          // fast class: work items to aim for (a multiple of the resident warps)
  uint32_t fast_warps;              // fast class: resident warps of k_fscore's persistent grid
};


// launchers (defined in the .cu files)
cudaError_t launch_stage(const CallArgs& a, cudaStream_t s);
cudaError_t launch_plan(const CallArgs& a, cudaStream_t s);
cudaError_t launch_seed(const CallArgs& a, cudaStream_t s);
cudaError_t launch_small(const CallArgs& a, cudaStream_t s);
typedef cudaError_t (*score_launcher_t)(const CallArgs& a, int nb_class, int grid, cudaStream_t s);
typedef cudaError_t (*fscore_launcher_t)(const CallArgs& a, int grid, cudaStream_t s);
cudaError_t launch_score(const CallArgs& a, int grid, cudaStream_t s);
int score_blocks_per_sm(int L, int nb_class);
struct SelectArgs {
  dyplan_batch in;
  const uint8_t* choice;   // [R*L*16]
  const uint8_t* status;   // [R*L]
  int32_t L;
  const int32_t* live;     // [B]
  int32_t* variant;        // [R]
  dyplan_bundle rescored;  // optional (pointers may be null)
  int32_t has_rescored;
};
cudaError_t launch_select(const SelectArgs& a, cudaStream_t s);
struct SwitchArgs {
  dyplan_batch in;
  dyplan_bundle bundle;            // choice, status, dom_model, corr64 (or corr)
  int32_t L;
  dyplan_switch_params p;
  const float* model_load;         // [M]
  const float* since_switch;       // [R]
  const uint32_t* dispatched;      // [R]
  int32_t* cur_variant;            // [R] in/out
  uint8_t* active_choice;          // [R*16] in/out
  uint8_t* switched;               // [R] out
};
cudaError_t launch_switch(const SwitchArgs& a, cudaStream_t s);

// ---- coefficient construction (dyplan_bind.cu) ----
struct BindArgs {
  dyplan_profiles prof;
  int32_t NN, KK;
  const int32_t* opt_off; const uint32_t* pred_mask; const uint8_t* skill; const uint8_t* role;
  const uint8_t* model; const uint8_t* backend; const uint8_t* policy;
  float* vuln; float* acc; int32_t* lat_us; float* cost; int32_t* demand;
};
cudaError_t launch_bind(const BindArgs& a, cudaStream_t s);

// ---- linear mode (dyplan_linear.cu) ----
constexpr int kLinHdrWords = 88;                        // LinHdr size in words
constexpr int kLinBlobWords = kLinHdrWords + 2 * (16 * 16 + 4);   // header + (w, d)[slot]
struct LinHdr {
  int32_t status;                 // DYPLAN_ST_OK / _INVALID / _TOO_LARGE
  int32_t n_orig, n_int;          // real nodes, nodes incl. dummies (>= 2)
  float jmag;                     // bound on the magnitude of J and of every partial sum of it, over the request's plans and the call's levels
  unsigned long long outer_total; // prod_{i>=3} K_i
  unsigned long long pad1;
  int32_t K[16];                  // options per internal node (1 for dummies)
  uint32_t succ[16];              // successor mask per node (all bits > i)
  int32_t optbase[16];            // first table slot of node i
  unsigned long long stride[16];  // canonical stride (0 for dummies)
};
static_assert(sizeof(LinHdr) == kLinHdrWords * 4, "LinHdr layout");
struct __align__(16) LinRec { float J; uint32_t pad; unsigned long long key; };   // an item's best per level
struct LinArgs {
  dyplan_batch in;
  dyplan_bundle out;
  dyplan_linear_extra extra;
  const float* cost;
  dyplan_linear_params p;
  int32_t L;
  float levels[DYPLAN_MAX_LEVELS];
  // scratch
  uint32_t* blob;                 // [R][kLinBlobWords]
  LinRec* rec;                    // [R*chunks*L] item records
  int32_t* gJ;                    // [R*L] best J published so far (order-preserving int encoding)
  uint32_t* counter;              // [2] dynamic work counters of the two passes
  uint32_t chunks;                // work items per request
  unsigned long long* plans;      // [1] total plans enumerated (stats)
};
cudaError_t launch_linear(const LinArgs& a, int grid, cudaStream_t s);

// ---- M0 issue-rate micro-benchmarks (dyplan_m0.cu) ----
int m0_count();
const char* m0_name(int op);
int m0_warps_per_block();
double m0_warp_inst_per_warp();
cudaError_t m0_launch(int op, int grid, long long* stamps, float* sink, cudaStream_t s);

__host__ __device__ inline int nb_class_of(int B, bool has_caps) { return !has_caps ? 0 : (B <= 2 ? 2 : (B <= 4 ? 4 : 8)); }

}  // namespace dyplan
