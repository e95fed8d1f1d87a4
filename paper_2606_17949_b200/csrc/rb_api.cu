// rb_api.cu -- the C ABI of include/routebalance.h: context, argument checking, buffer staging, the launch
// sequence of one decision (a0..a7) and its CUDA-graph replay (a9).  Every step of the path runs in the
// kernels of scan_tc.cu / estimate.cu / score_dispatch.cu; nothing here computes on the host.
#include "../../include/routebalance.h"
#include "../../include/routebalance_testing.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <unordered_map>
#include <utility>
#include <vector>

#include <cudaTypedefs.h>

#include "rb_internal.cuh"

using namespace rb;

struct rb_ctx {
  // problem
  int64_t N = 0;
  int d = 0, M = 0, k = 0, kc = 0, kcap = 0, ks = 0;   // kc = k + slack; kcap >= kc; ks = entries the scan keeps
  rb_options opt{};
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  int num_sms = 148;
  // bank
  void* bank = nullptr;          // what the tensor-core scan reads: bf16 [N x d], or (fp32 storage) the split bank bf16 [N x 3 d]
  float* bank32 = nullptr;       // fp32 storage: the fp32 bank [N x d] the exact re-rank reads
  int d_scan = 0;                // columns of a scanned row: d, or kSplitPlanes d (fp32 storage: two-plane bf16 split)
  float* bank_quality = nullptr; // [N x M]
  float* bank_outlen = nullptr;
  // instances
  int I = 0;
  int32_t *tier = nullptr, *cap = nullptr, *present = nullptr;
  float *price_in = nullptr, *price_out = nullptr, *pre = nullptr, *dec = nullptr, *slope = nullptr;
  float *dec_i = nullptr, *slope_i = nullptr;   // [I] per-instance copies of the tier coefficients
  float* dq = nullptr;
  int32_t* bq = nullptr;
  // per-call staging + scratch (sized by max_batch)
  int Bpad_max = 0;
  float* q32 = nullptr;             // [max_batch x d] fp32 storage: device copy of the queries for the exact re-rank
  float* q32_in = nullptr;          // [max_batch x d] staging of host queries that do not fit the pinned block
  __nv_bfloat16* qs = nullptr;      // [Bpad_max x d]
  int32_t* plen = nullptr;          // [max_batch]
  CallParams cp_cur{};              // per-call parameters of the call being enqueued (passed to the kernels by value)
  uint32_t* gthr = nullptr;         // [Bpad_max] cross-slab admission thresholds of the scan (cleared per decision)
  float* part_sim = nullptr;        // [num_sms][kcap][Bpad_max]
  int32_t* part_idx = nullptr;
  int32_t* scratch_nn_idx = nullptr;   // [max_batch x k] staging for host callers
  float* scratch_nn_sim = nullptr;
  float *pred_q = nullptr, *pred_l = nullptr;   // [max_batch x M] the estimate, consumed by score/dispatch
  float *stage_q = nullptr, *stage_l = nullptr; // [max_batch x M] staging of caller-supplied predictions (host)
  float *termA = nullptr, *termP = nullptr, *key = nullptr;
  // Pipelined decisions (rb_options.pipeline): a second set of everything a decision's estimate hands to its dispatch
  // side (staged queries + their tensor map, partial lists, predictions, terms, keys), internal streams for the staging
  // and for the scan, and the events that order the three parts of a decision and the reuse of a set.
  struct Slot {
    __nv_bfloat16* qs = nullptr;
    CUtensorMap tm_q{};
    float* part_sim = nullptr;
    int32_t* part_idx = nullptr;
    float *pred_q = nullptr, *pred_l = nullptr, *termA = nullptr, *termP = nullptr, *key = nullptr;
    float* q32 = nullptr;             // fp32 storage: this set's copy of the queries for the exact re-rank
    uint32_t* gthr = nullptr;         // the pair scan's cross-slab admission thresholds (cleared by the staging kernel)
    cudaEvent_t ev_stage = nullptr;   // staging done, recorded on the staging stream
    cudaEvent_t ev_front = nullptr;   // bank scan done, recorded on the front stream
    cudaEvent_t ev_back = nullptr;    // back half (finish + dispatch) done, recorded on the context's stream
  } slot[kSlots];
  cudaStream_t front = nullptr;       // low-priority internal stream of the bank scans
  cudaStream_t front2 = nullptr;      // second stream of the bank scans (see run_pipelined)
  cudaStream_t sstage = nullptr;      // internal stream of the staging kernels
  cudaEvent_t ev_bigfin = nullptr;    // finishing kernel of the last pipelined decision of more than 128 requests done
  bool bigfin_pending = false;        // ... and the next scan has not waited for it yet (they run beside the scan before them)
  uint64_t pipe_seq = 0;              // pipelined decisions issued so far (slot = seq % kSlots)
  bool front_busy = false;            // a front half may still be running on the internal stream
  int32_t *order = nullptr, *assignment = nullptr, *max_tokens = nullptr;
  float* budget = nullptr;          // [max_batch] staging of host budgets
  uint8_t* arena = nullptr;         // one allocation behind all the small per-decision buffers
  int32_t *members = nullptr, *tstart = nullptr, *pipe_cursor = nullptr;   // pipeline mode: tier membership, cursors
  unsigned long long* pipe_counter = nullptr;
  uint8_t* sweep_buf = nullptr;     // rb_sweep_weights: [P x 3] weights | [P][B x M] termA | termP | [P][B] key | assignment
  size_t sweep_cap = 0;
  // Host callers of rb_decide: inputs are copied (host memcpy) into this pinned block, which the kernels read over the
  // bus directly, and the assignment is written into it by the dispatch kernel -- no copy-engine transfers on the path.
  uint8_t* h_zc = nullptr;          // pinned host block: [query | plen | budget | assignment]
  uint8_t* d_zc = nullptr;          // the same block as the device addresses it
  size_t zc_query_cap = 0, zc_off_plen = 0, zc_off_budget = 0, zc_off_assign = 0, zc_off_flag = 0;
  uint32_t done_seq = 0;
  // rb_decide_submit / rb_decide_collect: one pinned block per buffer set ([query | plen | assignment | completion word],
  // at most 128 requests) and what is in flight in it
  struct AsyncSlot {
    uint8_t *h = nullptr, *d = nullptr;
    bool busy = false;
    uint32_t seq = 0;
    int B = 0;
  } async[kSlots];
  size_t az_off_plen = 0, az_off_assign = 0, az_off_flag = 0;
  uint64_t async_head = 0;            // submissions collected so far (the oldest in flight: the busy block with the smallest sequence number)
  uint64_t async_tail = 0;            // submissions made so far
  // boosted TPOT head (latency_mode 2)
  int4* f_nodes = nullptr;
  int32_t *f_root = nullptr, *f_begin = nullptr, *f_nbegin = nullptr;   // roots, trees per tier, nodes per tier
  uint32_t* f_cwords = nullptr;       // the packed forest (ForestDev::cwords) ...
  int32_t* f_cbegin = nullptr;        // ... and its per-tier blocks
  int f_total_cwords = 0, f_max_tier_cwords = 0;
  int f_max_tier_nodes = 0;
  float f_tpot_hi = 0.0f;             // bound of the head's output over all states (see ForestDev)
  float *f_base = nullptr, *f_aux = nullptr, *f_tpot0 = nullptr;
  int f_features = 0;
  bool has_forest = false;
  // rb_advance_state calls not yet applied on the device: the next rb_decide folds them into its first kernel
  float pending_adv[kMaxPendingAdvance]{};
  int n_pending = 0;
  float *scores = nullptr, *scores0 = nullptr;  // [max_batch x I], allocated by rb_set_instances
  CUtensorMap tm_q{}, tm_bank{}, tm_bank16{};   // bank: 64-row boxes; the same with 16-row boxes
  // graphs: key from (B, kind, buffer set, stage timing); kinds: 0 decide, 1 estimate, 2 from_predictions; throughput mode:
  // 5 staging, 3 scan, 4 finish + dispatch
  // One captured graph per decision shape.  The per-call parameters are an argument of the kernels that need them; a
  // replay rewrites that one argument of those kernel nodes (cudaGraphExecKernelNodeSetParams) -- no transfer of any
  // kind sits between the host and the decision's first kernel.
  struct CpNode {
    cudaGraphNode_t node;
    cudaKernelNodeParams params;
    std::vector<void*> args;   // the node's argument pointers, with args[cp_index] redirected to cp_cur
    int cp_index;
  };
  struct GraphRec {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    int nodes = 0;
    std::vector<CpNode> cp_nodes;
  };
  std::unordered_map<int64_t, GraphRec> graphs;
  int64_t launches = 0;
  bool stage_timing = false;
  bool capturing = false;
  cudaEvent_t ev[8]{};
  float stage_us[6]{};
  unsigned long long* dev_clock = nullptr;   // [2] scan kernel's earliest CTA start / latest CTA end (stage-timing mode)
  unsigned long long* dev_clock_init = nullptr;   // [2] = {~0, 0} in device memory
  float scan_device_us = 0.0f;
  std::string err;
};

namespace {


rb_status fail(rb_ctx* c, rb_status st, const char* what, cudaError_t e = cudaSuccess) {
  if (c) {
    char buf[512];
    if (e != cudaSuccess)
      snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    else
      snprintf(buf, sizeof buf, "%s", what);
    c->err = buf;
  }
  return st;
}

#define CK(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return fail(ctx, RB_ECUDA, #call, e_); \
  } while (0)

bool is_host_ptr(const void* p) {
  cudaPointerAttributes a{};
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return true;
  }
  return !(a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged);
}

template <typename T>
cudaError_t dev_alloc(T** p, size_t n) {
  return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T));
}

DispatchModes modes_of(const rb_ctx* c) {
  DispatchModes m;
  m.lpt_enabled = c->opt.lpt_enabled; m.update_mode = c->opt.update_enabled; m.tiebreak_mode = c->opt.tiebreak_mode;
  m.latency_mode = c->opt.latency_mode;
  return m;
}

ForestDev forest_of(const rb_ctx* c) {
  ForestDev f{};
  f.nodes = c->f_nodes; f.tree_root = c->f_root; f.tier_begin = c->f_begin; f.base = c->f_base; f.aux = c->f_aux;
  f.tpot0 = c->f_tpot0; f.n_features = c->f_features; f.tier_node_begin = c->f_nbegin; f.max_tier_nodes = c->f_max_tier_nodes; f.tpot_hi = c->f_tpot_hi;
  f.cwords = c->f_cwords; f.tier_cbegin = c->f_cbegin; f.total_cwords = c->f_total_cwords; f.max_tier_cwords = c->f_max_tier_cwords;
  return f;
}

void drop_graphs(rb_ctx* c) {
  for (auto& kv : c->graphs) {
    cudaGraphExecDestroy(kv.second.exec);
    cudaGraphDestroy(kv.second.graph);
  }
  c->graphs.clear();
}

InstTable table_of(const rb_ctx* c) {
  InstTable t;
  t.I = c->I; t.M = c->M; t.tier = c->tier; t.cap = c->cap; t.price_in = c->price_in; t.price_out = c->price_out;
  t.pre = c->pre; t.dec = c->dec; t.slope = c->slope; t.present = c->present; t.dec_i = c->dec_i; t.slope_i = c->slope_i;
  return t;
}

// Applies the pending rb_advance_state calls with the standalone kernel (every path but rb_decide's bf16 pipeline).
rb_status flush_pending(rb_ctx* ctx) {
  for (int a = 0; a < ctx->n_pending; ++a) {
    CK(launch_advance(table_of(ctx), ctx->dq, ctx->bq, ctx->pending_adv[a], ctx->stream));
    ctx->launches += 1;
  }
  ctx->n_pending = 0;
  return RB_OK;
}

rb_status encode_map(rb_ctx* ctx, CUtensorMap* map, void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
  if (!fn) {
    cudaDriverEntryPointQueryResult q;
    void* p = nullptr;
    CK(cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &p, 12000, cudaEnableDefault, &q));
    if (q != cudaDriverEntryPointSuccess || !p) return fail(ctx, RB_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    fn = (PFN_cuTensorMapEncodeTiled_v12000)p;
  }
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * 2};
  cuuint32_t box[2] = {(cuuint32_t)kTileK, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[96];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
    return fail(ctx, RB_ECUDA, buf);
  }
  return RB_OK;
}

bool finite_nonneg(float x) { return std::isfinite(x) && x >= 0.0f; }

rb_status check_weights(rb_ctx* ctx, const float w[3]) {
  if (!w) return fail(ctx, RB_EINVAL, "w is NULL");
  float sum = 0.0f;
  for (int j = 0; j < 3; ++j) {
    if (!finite_nonneg(w[j])) return fail(ctx, RB_EINVAL, "weights must be finite and >= 0");
    sum += w[j];
  }
  if (std::fabs(sum - 1.0f) > 1e-5f) return fail(ctx, RB_EINVAL, "weights must sum to 1 (3-simplex, P:L90)");
  return RB_OK;
}

// ---- the launch sequence ------------------------------------------------------------------------------
struct Timer {
  rb_ctx* c;
  int idx = 0;
  explicit Timer(rb_ctx* c_) : c(c_) {}
  void mark() {
    // (inside a capture the record becomes an event node of the graph; "external" keeps the event usable for timing)
    if (c->stage_timing) cudaEventRecordWithFlags(c->ev[idx++], c->stream, c->capturing ? cudaEventRecordExternal : cudaEventRecordDefault);
  }
};

// with_terms: the finishing kernel also derives the score terms (rb_decide); otherwise estimate only.
// sl: buffer set.  part: kAll = staging + scan + finish on stream s; kStage / kScan / kBack = one of the three
// (throughput mode: each on its own stream).
enum EstimatePart { kAll = 0, kStage = 1, kScan = 2, kBack = 3 };
rb_status enqueue_estimate(rb_ctx* ctx, int B, bool with_terms, Timer& tm, int sl = 0, EstimatePart part = kAll,
                           cudaStream_t s = nullptr) {
  if (!s) s = ctx->stream;
  rb_ctx::Slot& S = ctx->slot[sl];
  const int Bpad = (B + kTileM - 1) / kTileM * kTileM;
  FinishArgs fa{};
  fa.kc = ctx->kc; fa.k = ctx->k; fa.N = ctx->N; fa.d = ctx->d;
  fa.bank_quality = ctx->bank_quality; fa.bank_outlen = ctx->bank_outlen; fa.M = ctx->M;
  fa.weight_mode = ctx->opt.weight_mode; fa.eps = ctx->opt.dist_eps; fa.with_terms = with_terms ? 1 : 0;
  fa.pred_q = S.pred_q; fa.pred_l = S.pred_l; fa.termA = S.termA; fa.termP = S.termP; fa.key = S.key;
  const bool do_stage = part == kAll || part == kStage, do_scan = part == kAll || part == kScan, back = part == kAll || part == kBack;
  const bool front = do_stage || do_scan;
  const int split = ctx->opt.store_dtype == RB_F32 ? 1 : 0;   // fp32 storage: the scan runs over the three-plane bf16 split
  {
    if (ctx->stage_timing && front) {   // before the first mark: nothing but the kernels between the stage events
      CK(cudaMemcpyAsync(ctx->dev_clock, ctx->dev_clock_init, 16, cudaMemcpyDeviceToDevice, s));
    }
    if (front) tm.mark();
    if (B > kTileM && ctx->num_sms >= 2) {
      // tensor-bound regime: CTA pairs, 256-query m-tiles
      const int Bpad2 = (B + 2 * kTileM - 1) / (2 * kTileM) * (2 * kTileM);
      // throughput mode: one cluster's two SMs are left to the dispatch CTA of the decision before
      const int sms2 = (part != kAll && ctx->num_sms >= 64) ? ctx->num_sms - 2 : ctx->num_sms;
      const int ncl = scan_tc2_clusters(ctx->N, sms2);
      // lists of at most 32 entries per (cluster, query): 64-entry lists put the sorted insertions (in global memory) on
      // the tensor pipe's time line (k = 32: 0.54 of the tensor roofline), 16-entry ones under k + slack = 40 weaken the
      // pooled admission bound (0.69 against 0.74 with 32, C4 at B = 512 and 4096); a cluster whose list is popped
      // completely is searched again by the finishing kernel, as for the single-CTA scan
      const int kcap2 = std::min(ctx->kcap, 32);
      if (do_stage) {
        CK(launch_stage_queries(ctx->cp_cur, S.qs, B, Bpad2, ctx->d, 1, S.gthr, Bpad2 * (1 + ncl), split, S.q32, s));
        tm.mark();
        ctx->launches += 1;
      }
      if (do_scan) {
        int ncl_used = 0;
        CK(launch_scan_tc2(&S.tm_q, &ctx->tm_bank, ctx->N, ctx->d_scan, B, Bpad2, kcap2, ctx->kc, sms2, S.part_sim, S.part_idx,
                           S.gthr, &ncl_used, s));
        tm.mark();
        ctx->launches += 1;
      }
      fa.part_sim = S.part_sim; fa.part_idx = S.part_idx; fa.nlists = ncl; fa.lists_per_cta = 1; fa.kcap = kcap2;
      fa.Bpad = Bpad2; fa.slab_unit = kTileN; fa.rescan = kcap2 < ctx->kc ? 1 : 0;
    } else {
      const int rep = scan_tc_replicas(B, ctx->ks, ctx->num_sms);
      const int64_t units = (ctx->N + kBoxN - 1) / kBoxN;
      // Throughput mode: the scan leaves a few SMs to the back half of the decision before it (one finishing CTA per
      // request, then the dispatch CTA), which otherwise waits for scan CTAs to leave and delays the scan CTAs that come
      // after it.  Measured on B200 (C2, decisions back to back): B = 11: 38.9 -> 33.1 us per decision with 12 SMs kept
      // free, B = 32: 42.9 -> 34.3 with 32, B = 64: 51.8 -> 40.4 with 16 (more costs the scan more than it saves).
      int sms = ctx->num_sms;
      if (part != kAll && ctx->num_sms >= 64) sms -= B <= 32 ? (B + 3) / 4 * 4 : 16;
      const int grid = (int)(units < sms ? units : sms);   // what launch_scan_tc uses
      if (do_stage) {
        CK(launch_stage_queries(ctx->cp_cur, S.qs, B, Bpad, ctx->d, rep, ctx->gthr, 0, split, S.q32, s));
        tm.mark();
        ctx->launches += 1;
      }
      if (do_scan) {
        int grid_used = 0;
        CK(launch_scan_tc(&S.tm_q, &ctx->tm_bank, &ctx->tm_bank16, ctx->N, ctx->d_scan, B, Bpad, ctx->ks, sms, S.part_sim, S.part_idx,
                          &grid_used, ctx->stage_timing ? ctx->dev_clock : nullptr, s));
        tm.mark();
        ctx->launches += 1;
      }
      fa.part_sim = S.part_sim; fa.part_idx = S.part_idx; fa.nlists = grid * rep; fa.lists_per_cta = rep; fa.kcap = ctx->ks;
      fa.records = 1;
      fa.Bpad = Bpad; fa.slab_unit = kRowUnit;
      fa.rescan = ctx->ks < ctx->kc ? 1 : 0;
    }
    if (split) {   // exact similarities from the fp32 rows (the definition of fp32 storage), always
      fa.bank = nullptr; fa.qs = nullptr; fa.bank32 = ctx->bank32; fa.q32 = S.q32; fa.rerank = 2;
    } else {
      fa.bank = (const __nv_bfloat16*)ctx->bank; fa.qs = S.qs; fa.rerank = ctx->opt.rerank_slack > 0 ? 1 : 0;
    }
  }
  if (back) {
    CK(launch_finish(fa, table_of(ctx), ctx->cp_cur, B, s));
    ctx->launches += 1;
    tm.mark();
  }
  return RB_OK;
}

rb_status enqueue_dispatch(rb_ctx* ctx, int B, bool from_predictions, Timer& tm, int sl = 0) {
  cudaStream_t s = ctx->stream;
  rb_ctx::Slot& S = ctx->slot[sl];
  InstTable t = table_of(ctx);
  if (from_predictions) {
    if (ctx->opt.latency_mode == 2) {
      CK(launch_tpot_forest(t, forest_of(ctx), ctx->dq, ctx->bq, ctx->f_tpot0, -1.0f, s));
      ctx->launches += 1;
    }
    CK(launch_score(t, ctx->dq, ctx->bq, ctx->cp_cur, B, S.termA, S.termP, S.key, modes_of(ctx), forest_of(ctx), s));
    ctx->launches += 1;
  }
  tm.mark();
  CK(launch_lpt_dispatch(t, ctx->dq, ctx->bq, S.termA, S.termP, S.key, ctx->cp_cur, B, modes_of(ctx), forest_of(ctx), s));
  tm.mark();
  ctx->launches += 1;
  return RB_OK;
}

// Runs the launch sequence `enqueue` on stream s as a CUDA graph: captured and instantiated the first time a key is seen,
// replayed afterwards with this call's parameters (the per-call parameters are an argument of the kernels that need them;
// a replay rewrites that one argument of those kernel nodes, cudaGraphExecKernelNodeSetParams).
template <typename F>
rb_status graph_run(rb_ctx* ctx, int64_t gkey, cudaStream_t s, F&& enqueue) {
  auto it = ctx->graphs.find(gkey);
  if (it == ctx->graphs.end()) {
    const int64_t before = ctx->launches;
    cudaGraph_t g = nullptr;
    CK(cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
    ctx->capturing = true;
    rb_status st = enqueue();
    cudaError_t e = cudaStreamEndCapture(s, &g);
    ctx->capturing = false;
    const int nodes = (int)(ctx->launches - before);
    ctx->launches = before;
    if (st != RB_OK) {
      if (g) cudaGraphDestroy(g);
      return st;
    }
    if (e != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaStreamEndCapture", e);
    rb_ctx::GraphRec rec;
    rec.graph = g;
    rec.nodes = nodes;
    e = cudaGraphInstantiate(&rec.exec, g, 0);
    if (e != cudaSuccess) {
      cudaGraphDestroy(g);
      return fail(ctx, RB_ECUDA, "cudaGraphInstantiate", e);
    }
    // the kernel nodes that take the per-call parameters, and where
    size_t nn = 0;
    CK(cudaGraphGetNodes(g, nullptr, &nn));
    std::vector<cudaGraphNode_t> all(nn);
    CK(cudaGraphGetNodes(g, all.data(), &nn));
    for (cudaGraphNode_t node : all) {
      cudaGraphNodeType ty;
      CK(cudaGraphNodeGetType(node, &ty));
      if (ty != cudaGraphNodeTypeKernel) continue;
      rb_ctx::CpNode cn{};
      CK(cudaGraphKernelNodeGetParams(node, &cn.params));
      int nargs = 0;
      int idx = estimate_cp_arg(cn.params.func, &nargs);
      if (idx < 0) idx = dispatch_cp_arg(cn.params.func, &nargs);
      if (idx < 0) continue;
      cn.node = node;
      cn.cp_index = idx;
      cn.args.assign(cn.params.kernelParams, cn.params.kernelParams + nargs);   // values stay owned by the node
      rec.cp_nodes.push_back(std::move(cn));
    }
    it = ctx->graphs.emplace(gkey, std::move(rec)).first;
  } else {
    // replay: the same graph with this call's parameters
    for (rb_ctx::CpNode& cn : it->second.cp_nodes) {
      cn.args[cn.cp_index] = &ctx->cp_cur;
      cn.params.kernelParams = cn.args.data();
      CK(cudaGraphExecKernelNodeSetParams(it->second.exec, cn.node, &cn.params));
    }
  }
  CK(cudaGraphLaunch(it->second.exec, s));
  ctx->launches += it->second.nodes;
  return RB_OK;
}

int64_t graph_key(const rb_ctx* ctx, int B, int kind, int sl) {
  return (((int64_t)B * 8 + kind) * kSlots + sl) * 2 + (ctx->stage_timing ? 1 : 0);
}

// kind: 0 = estimate + dispatch, 1 = estimate, 2 = dispatch (+scores0)
rb_status run_path(rb_ctx* ctx, int B, int kind) {
  // With stage timing on, the same launch sequence is captured with event-record nodes between the kernels (a
  // separate graph per shape): the stage intervals then hold graph-internal launch latencies like a decision's, not
  // host-side ones.  The kernels lose their programmatic overlap across the event nodes, so the SUM of the stages is
  // longer than a decision; each stage's own duration is what is read.
  Timer tm(ctx);
  auto enqueue = [&]() -> rb_status {
    if (kind == 0 && ctx->opt.latency_mode == 2) {   // the head over the batch-start state; only the state feeds it
      if (launch_tpot_forest(table_of(ctx), forest_of(ctx), ctx->dq, ctx->bq, ctx->f_tpot0, -1.0f, ctx->stream) != cudaSuccess)
        return fail(ctx, RB_ECUDA, "launch_tpot_forest");
      ctx->launches += 1;
    }
    rb_status st = RB_OK;
    if (kind != 2) st = enqueue_estimate(ctx, B, kind == 0, tm);
    if (st == RB_OK && kind != 1) st = enqueue_dispatch(ctx, B, kind == 2, tm);
    return st;
  };
  rb_status st = ctx->opt.use_graph ? graph_run(ctx, graph_key(ctx, B, kind, 0), ctx->stream, enqueue) : enqueue();
  // (a later pipelined decision's front half must not start on this buffer set before this work is done)
  if (st == RB_OK && ctx->front && kind != 2) CK(cudaEventRecord(ctx->slot[0].ev_back, ctx->stream));
  return st;
}

// rb_decide in throughput mode (rb_options.pipeline): the bank scan goes to one of two internal low-priority streams
// (consecutive decisions alternate); the query staging in front of it to a second internal stream, so
// that it runs beside the scan of the decision before (C2, B = 11: 33.1 -> 31.0 us per decision); the back half
// (finishing + dispatch) to the context's stream.  Events join the three; kSlots buffer sets rotate
// (three: with two, the scan of decision j + 2 waits for the back half of decision j, and a host loop of submissions is
// limited to two in flight, i.e. to half a decision's latency per decision).
rb_status run_pipelined(rb_ctx* ctx, int B) {
  const int sl = (int)(ctx->pipe_seq % kSlots);
  rb_ctx::Slot& S = ctx->slot[sl];
  Timer tm(ctx);
  // The scans of consecutive decisions alternate between two streams: the CTAs of scan j + 1 start on the SMs that the
  // CTAs of scan j leave (its slabs end up to 3.7 us apart), instead of behind a kernel boundary and a launch gap -- C2,
  // decisions back to back, B = 11: 30.9 -> 23.8 us per decision, B = 64: 42 -> 34.  (Two scans under way read the same
  // bank a few MB apart, so part of the later one's lines come from L2: 23.8 us is less than one scan alone takes.)
  // Staging: beside the scan of the decision before (on the SMs that scan leaves free), once the back half that last
  // read this buffer set is done.
  cudaStream_t fr = (ctx->pipe_seq & 1) ? ctx->front2 : ctx->front;
  cudaStream_t sstage = ctx->sstage;
  CK(cudaStreamWaitEvent(sstage, S.ev_back, 0));
  rb_status st = graph_run(ctx, graph_key(ctx, B, 5, sl), sstage,
                           [&]() -> rb_status { return enqueue_estimate(ctx, B, true, tm, sl, kStage, sstage); });
  if (st != RB_OK) return st;
  CK(cudaEventRecord(S.ev_stage, sstage));
  CK(cudaStreamWaitEvent(fr, S.ev_stage, 0));
  if (ctx->bigfin_pending) {
    // the decision before has more than 128 requests: its finishing kernel (one CTA per request) wants the whole GPU, so
    // this scan starts behind it -- and then runs beside that decision's dispatch CTA
    CK(cudaStreamWaitEvent(fr, ctx->ev_bigfin, 0));
    ctx->bigfin_pending = false;
  }
  st = graph_run(ctx, graph_key(ctx, B, 3, sl), fr,
                 [&]() -> rb_status { return enqueue_estimate(ctx, B, true, tm, sl, kScan, fr); });
  if (st != RB_OK) return st;
  CK(cudaEventRecord(S.ev_front, fr));
  CK(cudaStreamWaitEvent(ctx->stream, S.ev_front, 0));
  if (B > kTileM) {
    st = graph_run(ctx, graph_key(ctx, B, 4, sl), ctx->stream,
                   [&]() -> rb_status { return enqueue_estimate(ctx, B, true, tm, sl, kBack, ctx->stream); });
    if (st != RB_OK) return st;
    CK(cudaEventRecord(ctx->ev_bigfin, ctx->stream));
    ctx->bigfin_pending = true;
    st = graph_run(ctx, graph_key(ctx, B, 6, sl), ctx->stream,
                   [&]() -> rb_status { return enqueue_dispatch(ctx, B, false, tm, sl); });
  } else {
    st = graph_run(ctx, graph_key(ctx, B, 4, sl), ctx->stream, [&]() -> rb_status {
      rb_status s1 = enqueue_estimate(ctx, B, true, tm, sl, kBack, ctx->stream);
      return s1 != RB_OK ? s1 : enqueue_dispatch(ctx, B, false, tm, sl);
    });
  }
  if (st != RB_OK) return st;
  CK(cudaEventRecord(S.ev_back, ctx->stream));
  ctx->pipe_seq += 1;
  return RB_OK;
}

void collect_stage_times(rb_ctx* ctx, int kind) {
  if (!ctx->stage_timing) return;
  cudaStreamSynchronize(ctx->stream);
  for (float& v : ctx->stage_us) v = 0.0f;
  {
    unsigned long long h[2] = {0, 0};
    ctx->scan_device_us = 0.0f;
    if (cudaMemcpy(h, ctx->dev_clock, sizeof h, cudaMemcpyDeviceToHost) == cudaSuccess && h[1] > h[0] && h[0] != ~0ull)
      ctx->scan_device_us = (float)((double)(h[1] - h[0]) * 1e-3);
  }
  auto span = [&](int e0, int e1) {
    float ms = 0;
    return cudaEventElapsedTime(&ms, ctx->ev[e0], ctx->ev[e1]) == cudaSuccess ? ms * 1000.0f : 0.0f;
  };
  // marks: estimate = 4 events (stage | scan | merge+aggregate), then dispatch = 2 more (score | dispatch)
  if (kind != 2) {
    ctx->stage_us[0] = span(0, 1);
    ctx->stage_us[1] = span(1, 2);
    ctx->stage_us[3] = span(2, 3);   // merge is fused into the finishing kernel: reported under "aggregate"
    if (kind == 0) {
      ctx->stage_us[4] = span(3, 4);
      ctx->stage_us[5] = span(4, 5);
    }
  } else {
    ctx->stage_us[5] = span(0, 1);   // no mark precedes the score kernel: only the dispatch interval is known
  }
}

// The call's parameters: kept in the context while its kernels are enqueued (they receive them by value).
rb_status push_params(rb_ctx* ctx, const CallParams& cp) {
  ctx->cp_cur = cp;
  return RB_OK;
}

// Resolves caller buffers into device pointers for the parameter block.  Host inputs are copied into the
// context's staging buffer first; host outputs are produced in the staging buffer and copied back after the
// kernels (Stager::finish).
struct Stager {
  rb_ctx* ctx;
  bool any_host = false;
  bool wait_flag = false;    // completion is signalled through the pinned word (no stream synchronisation needed)
  bool needs_sync = false;   // some host buffer went through the copy engine: the stream must drain
  // classified on every call (cudaPointerGetAttributes): an address can change its memory kind between calls
  bool host(const void* p) { return is_host_ptr(p); }
  cudaError_t err = cudaSuccess;
  struct Back { void* dst; const void* src; size_t bytes; };
  Back back[10];
  int nback = 0;
  Back hback[2];   // host memcpys out of the pinned block, after the stream has drained
  int nhback = 0;
  // host input of at most `cap` bytes -> pinned block at `off`, read by the kernels in place
  template <typename T>
  const T* in_zc(const T* user, size_t off, size_t cap, T* staging, size_t bytes) {
    if (!host(user)) return user;
    if (ctx->h_zc == nullptr || bytes > cap) return in(user, staging, bytes);
    any_host = true;
    std::memcpy(ctx->h_zc + off, user, bytes);
    return reinterpret_cast<const T*>(ctx->d_zc + off);
  }
  template <typename T>
  T* out_zc(T* user, size_t off, T* staging, size_t bytes) {
    if (!user) return nullptr;
    if (!host(user)) return user;
    if (ctx->h_zc == nullptr) return out(user, staging, bytes);
    any_host = true;
    wait_flag = true;
    hback[nhback++] = Back{user, ctx->h_zc + off, bytes};
    return reinterpret_cast<T*>(ctx->d_zc + off);
  }
  template <typename T>
  const T* in(const T* user, T* staging, size_t bytes) {
    if (!host(user)) return user;
    any_host = true;
    needs_sync = true;
    if (err == cudaSuccess) err = cudaMemcpyAsync(staging, user, bytes, cudaMemcpyHostToDevice, ctx->stream);
    return staging;
  }
  template <typename T>
  T* out(T* user, T* staging, size_t bytes) {
    if (!user) return nullptr;
    if (!host(user)) return user;
    any_host = true;
    needs_sync = true;
    back[nback++] = Back{user, staging, bytes};
    return staging;
  }
  // an output that the kernels always produce in `internal`: device callers get an extra copy through the
  // parameter block, host callers a D2H copy afterwards
  template <typename T>
  T* out_internal(T* user, T* internal, size_t bytes) {
    if (!user) return nullptr;
    if (!host(user)) return user;
    any_host = true;
    needs_sync = true;
    back[nback++] = Back{user, internal, bytes};
    return nullptr;
  }
  rb_status finish() {
    for (int j = 0; j < nback && err == cudaSuccess; ++j)
      err = cudaMemcpyAsync(back[j].dst, back[j].src, back[j].bytes, cudaMemcpyDeviceToHost, ctx->stream);
    if (err != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaMemcpyAsync (outputs)", err);
    // host-side inputs must be consumed and host-side outputs complete before returning
    if (any_host) {
      if (wait_flag && !needs_sync) {
        // the dispatch kernel stores the call's sequence number into the pinned word after the assignment: poll it
        // (a stream synchronisation costs several microseconds more); the stream is queried now and then so that
        // a failed launch cannot hang the caller
        volatile uint32_t* flag = reinterpret_cast<volatile uint32_t*>(ctx->h_zc + ctx->zc_off_flag);
        for (uint32_t spins = 1; *flag != ctx->done_seq; ++spins) {
          if ((spins & 0x3fff) == 0) {
            const cudaError_t q = cudaStreamQuery(ctx->stream);
            if (q == cudaSuccess) break;
            if (q != cudaErrorNotReady) return fail(ctx, RB_ECUDA, "cudaStreamQuery", q);
          }
        }
        if (*flag != ctx->done_seq) CK(cudaStreamSynchronize(ctx->stream));
      } else {
        CK(cudaStreamSynchronize(ctx->stream));
      }
    }
    for (int j = 0; j < nhback; ++j) std::memcpy(hback[j].dst, hback[j].src, hback[j].bytes);
    return RB_OK;
  }
};

}  // namespace

extern "C" {

void rb_options_default(rb_options* opt) {
  if (!opt) return;
  std::memset(opt, 0, sizeof *opt);
  opt->bank_dtype = RB_F32;
  opt->store_dtype = RB_BF16;
  opt->weight_mode = 0;
  opt->dist_eps = 1e-6f;
  opt->rerank_slack = 6;
  opt->lpt_enabled = 1;
  opt->update_enabled = 1;
  opt->max_batch = 4096;
  opt->use_graph = 1;
  opt->scan_list = 0;
  opt->tiebreak_mode = 0;
  opt->latency_mode = 0;
  opt->pipeline = 0;
  opt->stream = nullptr;
}

rb_status rb_create(rb_ctx** out, const void* bank_emb, const float* bank_quality, const float* bank_outlen, int64_t N,
                    int32_t d, int32_t M, int32_t k, const rb_options* opt_in) {
  if (!out) return RB_EINVAL;
  *out = nullptr;
  rb_options opt;
  if (opt_in) opt = *opt_in; else rb_options_default(&opt);
  if (!bank_emb || !bank_quality || !bank_outlen) return RB_EINVAL;
  if (N < 1 || N >= (int64_t)1 << 31 || d < 8 || d % 8 != 0 || M < 1 || M > kMaxM || k < 1 || k > N) return RB_EINVAL;
  if (opt.bank_dtype != RB_F32 && opt.bank_dtype != RB_BF16) return RB_EINVAL;
  if (opt.store_dtype != RB_F32 && opt.store_dtype != RB_BF16) return RB_EINVAL;
  if (opt.store_dtype == RB_F32 && opt.bank_dtype != RB_F32) return RB_EINVAL;
  if (opt.rerank_slack < 0) opt.rerank_slack = 0;
  // fp32 storage always re-ranks (exact fp32-row similarities are its definition): the candidates come from a scan of
  // the three-plane bf16 split, good to ~5e-6, so a few spare candidates are kept
  if (opt.store_dtype == RB_F32 && opt.rerank_slack == 0) opt.rerank_slack = std::min(6, kMaxK - k);
  if (k + opt.rerank_slack > kMaxK) return RB_EINVAL;
  if (opt.max_batch < 1 || opt.max_batch > 4096) return RB_EINVAL;
  if (!(opt.dist_eps >= 0.0f) || !std::isfinite(opt.dist_eps)) return RB_EINVAL;
  if (opt.weight_mode != 0 && opt.weight_mode != 1) return RB_EINVAL;
  if (opt.update_enabled < 0 || opt.update_enabled > 2) return RB_EINVAL;
  if (opt.tiebreak_mode != 0 && opt.tiebreak_mode != 1) return RB_EINVAL;
  if (opt.latency_mode < 0 || opt.latency_mode > 2) return RB_EINVAL;
  opt.lpt_enabled = opt.lpt_enabled ? 1 : 0;
  opt.pipeline = opt.pipeline ? 1 : 0;
  if (opt.scan_list != 0 && opt.scan_list != 4 && opt.scan_list != 8 && opt.scan_list != 16 && opt.scan_list != 32 &&
      opt.scan_list != 64)
    return RB_EINVAL;

  int dev = 0;
  cudaDeviceProp prop{};
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return RB_EUNSUPPORTED;
  }
  if (prop.major != 10) return RB_EUNSUPPORTED;   // sm_100a kernels only; there is no fallback path

  rb_ctx* ctx = new (std::nothrow) rb_ctx();
  if (!ctx) return RB_ENOMEM;
  ctx->N = N; ctx->d = d; ctx->M = M; ctx->k = k; ctx->opt = opt;
  ctx->d_scan = opt.store_dtype == RB_F32 ? kSplitPlanes * d : d;
  ctx->kc = k + opt.rerank_slack;
  ctx->kcap = ctx->kc <= 16 ? 16 : (ctx->kc <= 32 ? 32 : 64);
  ctx->num_sms = prop.multiProcessorCount;
  {
    // Entries the scan keeps per (CTA, query).  Short lists make the scan's warm-up cheap (its cost is in the
    // first few hundred rows of a slab); the finishing kernel searches a slab again, exactly, in the rare case
    // that a short list may hide members of the top kc.  Long slabs amortise a full-length list.
    const int64_t units = (N + kBoxN - 1) / kBoxN;
    const int64_t grid = units < ctx->num_sms ? units : ctx->num_sms;
    const int64_t rows_per_cta = N / grid;
    int ks = opt.scan_list;
    // (long slabs amortise the warm-up of a longer list, but past 16 entries the lock-step insertions of an
    // epilogue warp -- about KS*ln(rows/KS) per query, each ~6*KS instructions -- outgrow the time a tile's bytes take)
    if (ks == 0) ks = rows_per_cta >= 16384 ? std::min(ctx->kcap, 16) : (rows_per_cta >= 2048 ? 8 : 4);
    if (ks > ctx->kcap) ks = ctx->kcap;
    ctx->ks = ks;
  }
  ctx->Bpad_max = opt.max_batch <= kTileM ? kTileM : (opt.max_batch + 2 * kTileM - 1) / (2 * kTileM) * (2 * kTileM);
  *out = ctx;   // from here on errors keep the context so that rb_last_error works; caller destroys it

  if (opt.stream) {
    ctx->stream = (cudaStream_t)opt.stream;
  } else {
    CK(cudaStreamCreateWithFlags(&ctx->stream, cudaStreamNonBlocking));
    ctx->own_stream = true;
  }
  for (auto& e : ctx->ev) CK(cudaEventCreate(&e));
  {
    const size_t mbz = (size_t)opt.max_batch;
    ctx->zc_query_cap = std::min<size_t>(mbz * d * 4, (size_t)1 << 20);
    ctx->zc_off_plen = (ctx->zc_query_cap + 255) & ~(size_t)255;
    ctx->zc_off_budget = ctx->zc_off_plen + ((mbz * 4 + 255) & ~(size_t)255);
    ctx->zc_off_assign = ctx->zc_off_budget + ((mbz * 4 + 255) & ~(size_t)255);
    ctx->zc_off_flag = ctx->zc_off_assign + ((mbz * 4 + 255) & ~(size_t)255);
    const size_t total = ctx->zc_off_flag + 256;
    if (cudaHostAlloc((void**)&ctx->h_zc, total, cudaHostAllocMapped) == cudaSuccess &&
        cudaHostGetDevicePointer((void**)&ctx->d_zc, ctx->h_zc, 0) == cudaSuccess) {
      std::memset(ctx->h_zc, 0, total);
    } else {   // no mapped pinned memory: host callers go through the copy engine
      cudaGetLastError();
      if (ctx->h_zc) cudaFreeHost(ctx->h_zc);
  for (auto& A : ctx->async)
    if (A.h) cudaFreeHost(A.h);
      ctx->h_zc = nullptr;
      ctx->d_zc = nullptr;
    }
  }
  CK(cudaMalloc((void**)&ctx->dev_clock, 32));
  ctx->dev_clock_init = ctx->dev_clock + 2;
  {
    const unsigned long long init[4] = {0ull, 0ull, ~0ull, 0ull};
    CK(cudaMemcpy(ctx->dev_clock, init, sizeof init, cudaMemcpyHostToDevice));
  }
  cudaStream_t s = ctx->stream;
  const size_t nd = (size_t)N * d;
#define ALLOC(ptr, n)                                                                 \
  do {                                                                                \
    cudaError_t e_ = dev_alloc(&(ptr), (n));                                          \
    if (e_ != cudaSuccess) { cudaGetLastError(); return fail(ctx, RB_ENOMEM, "cudaMalloc " #ptr, e_); } \
  } while (0)

  if (opt.store_dtype == RB_BF16) {
    __nv_bfloat16* b16 = nullptr;
    ALLOC(b16, nd);
    ctx->bank = b16;
    if (opt.bank_dtype == RB_BF16) {
      CK(cudaMemcpyAsync(b16, bank_emb, nd * 2, cudaMemcpyDefault, s));
    } else {
      // fp32 -> bf16 (RNE) once, in chunks through a bounded device buffer
      const size_t chunk_rows = std::max<size_t>(1, ((size_t)64 << 20) / (size_t)d);
      float* tmp = nullptr;
      ALLOC(tmp, std::min<size_t>(chunk_rows, (size_t)N) * d);
      for (size_t r0 = 0; r0 < (size_t)N; r0 += chunk_rows) {
        const size_t rows = std::min(chunk_rows, (size_t)N - r0);
        CK(cudaMemcpyAsync(tmp, (const float*)bank_emb + r0 * d, rows * d * 4, cudaMemcpyDefault, s));
        CK(launch_convert_bf16(tmp, b16 + r0 * d, rows * d, s));
      }
      CK(cudaStreamSynchronize(s));
      cudaFree(tmp);
    }
  } else {
    // fp32 storage: the fp32 rows (exact re-rank) and their two-plane bf16 split in three column blocks (what the tensor cores scan)
    ALLOC(ctx->bank32, nd);
    CK(cudaMemcpyAsync(ctx->bank32, bank_emb, nd * 4, cudaMemcpyDefault, s));
    __nv_bfloat16* bs = nullptr;
    ALLOC(bs, kSplitPlanes * nd);
    ctx->bank = bs;
    CK(launch_split_bank(ctx->bank32, bs, (size_t)N, d, s));
  }
  ALLOC(ctx->bank_quality, (size_t)N * M);
  ALLOC(ctx->bank_outlen, (size_t)N * M);
  CK(cudaMemcpyAsync(ctx->bank_quality, bank_quality, (size_t)N * M * 4, cudaMemcpyDefault, s));
  CK(cudaMemcpyAsync(ctx->bank_outlen, bank_outlen, (size_t)N * M * 4, cudaMemcpyDefault, s));

  const size_t mb = opt.max_batch;
  ALLOC(ctx->q32, mb * d);
  ALLOC(ctx->q32_in, mb * d);
  // Everything a decision's latency-bound kernels touch (per-call parameters, instance table, state, per-request
  // terms and outputs) lives in ONE allocation, packed: a cold kernel then pays for one or two TLB misses instead
  // of one per buffer.
  {
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off = (off + bytes + 255) & ~(size_t)255; return o; };
    const size_t o_plen = take(mb * 4), o_pq = take(mb * M * 4), o_pl = take(mb * M * 4), o_sq = take(mb * M * 4),
                 o_sl = take(mb * M * 4), o_ta = take(mb * M * 4), o_tp = take(mb * M * 4), o_key = take(mb * 4),
                 o_ord = take(mb * 4), o_asg = take(mb * 4), o_mt = take(mb * 4), o_bud = take(mb * 4),
                 o_tier = take(kMaxI * 4), o_cap = take(kMaxI * 4), o_dq = take(kMaxI * 4), o_bq = take(kMaxI * 4),
                 o_pres = take(kMaxM * 4), o_pin = take(kMaxM * 4), o_pout = take(kMaxM * 4), o_pre = take(kMaxM * 4),
                 o_dec = take(kMaxM * 4), o_slope = take(kMaxM * 4), o_deci = take(kMaxI * 4), o_slopei = take(kMaxI * 4),
                 o_aux = take((size_t)kMaxI * kMaxFeatures * 4), o_tpot0 = take(kMaxI * 4), o_mem = take(kMaxI * 4),
                 o_tst = take((kMaxM + 1) * 4), o_cur = take(kMaxM * 4), o_cnt = take(8);
    // further sets of what an estimate hands to its dispatch side (pipelined decisions)
    const size_t m1 = opt.pipeline ? mb : 0;
    size_t o_pq1[kSlots], o_pl1[kSlots], o_ta1[kSlots], o_tp1[kSlots], o_key1[kSlots];
    for (int j = 1; j < kSlots; ++j) {
      o_pq1[j] = take(m1 * M * 4); o_pl1[j] = take(m1 * M * 4); o_ta1[j] = take(m1 * M * 4); o_tp1[j] = take(m1 * M * 4);
      o_key1[j] = take(m1 * 4);
    }
    ALLOC(ctx->arena, off);
    uint8_t* a = ctx->arena;
    ctx->plen = (int32_t*)(a + o_plen); ctx->pred_q = (float*)(a + o_pq); ctx->pred_l = (float*)(a + o_pl);
    ctx->stage_q = (float*)(a + o_sq); ctx->stage_l = (float*)(a + o_sl); ctx->termA = (float*)(a + o_ta);
    ctx->termP = (float*)(a + o_tp); ctx->key = (float*)(a + o_key); ctx->order = (int32_t*)(a + o_ord);
    ctx->assignment = (int32_t*)(a + o_asg); ctx->max_tokens = (int32_t*)(a + o_mt); ctx->budget = (float*)(a + o_bud);
    ctx->tier = (int32_t*)(a + o_tier); ctx->cap = (int32_t*)(a + o_cap); ctx->dq = (float*)(a + o_dq);
    ctx->bq = (int32_t*)(a + o_bq); ctx->present = (int32_t*)(a + o_pres); ctx->price_in = (float*)(a + o_pin);
    ctx->price_out = (float*)(a + o_pout); ctx->pre = (float*)(a + o_pre); ctx->dec = (float*)(a + o_dec);
    ctx->slope = (float*)(a + o_slope); ctx->dec_i = (float*)(a + o_deci); ctx->slope_i = (float*)(a + o_slopei);
    ctx->f_aux = (float*)(a + o_aux); ctx->f_tpot0 = (float*)(a + o_tpot0);
    ctx->members = (int32_t*)(a + o_mem); ctx->tstart = (int32_t*)(a + o_tst); ctx->pipe_cursor = (int32_t*)(a + o_cur);
    ctx->pipe_counter = (unsigned long long*)(a + o_cnt);
    for (int j = 1; j < kSlots; ++j) {
      rb_ctx::Slot& S1 = ctx->slot[j];
      S1.pred_q = (float*)(a + o_pq1[j]); S1.pred_l = (float*)(a + o_pl1[j]); S1.termA = (float*)(a + o_ta1[j]);
      S1.termP = (float*)(a + o_tp1[j]); S1.key = (float*)(a + o_key1[j]);
    }
    CK(cudaMemsetAsync(ctx->arena, 0, off, s));
  }
  {
    const int ds = ctx->d_scan;
    ALLOC(ctx->qs, (size_t)ctx->Bpad_max * ds);
    ALLOC(ctx->gthr, (size_t)ctx->Bpad_max * (2 + ctx->num_sms / 2));
    // [grid * rep][Bpad][ks]: rep = 4 replicas only when Bpad = 128
    const size_t part_n = (size_t)ctx->num_sms * ctx->kcap * std::max<size_t>(ctx->Bpad_max, 4 * kTileM);
    ALLOC(ctx->part_sim, 2 * part_n);          // one allocation: [similarities | indices], or 32-byte records over all of it
    ctx->part_idx = reinterpret_cast<int32_t*>(ctx->part_sim + part_n);
    CK(cudaMemsetAsync(ctx->qs, 0, (size_t)ctx->Bpad_max * ds * 2, s));
    rb_status st = encode_map(ctx, &ctx->tm_bank, ctx->bank, (uint64_t)N, (uint64_t)ds, kBoxN);
    if (st != RB_OK) return st;
    st = encode_map(ctx, &ctx->tm_bank16, ctx->bank, (uint64_t)N, (uint64_t)ds, kRowUnit);
    if (st != RB_OK) return st;
    st = encode_map(ctx, &ctx->tm_q, ctx->qs, (uint64_t)ctx->Bpad_max, (uint64_t)ds, kTileM);
    if (st != RB_OK) return st;
    if (opt.pipeline) {
      // further buffer sets, sized like the first
      for (int j = 1; j < kSlots; ++j) {
        rb_ctx::Slot& S1 = ctx->slot[j];
        ALLOC(S1.qs, (size_t)ctx->Bpad_max * ds);
        ALLOC(S1.part_sim, 2 * part_n);
        S1.part_idx = reinterpret_cast<int32_t*>(S1.part_sim + part_n);
        ALLOC(S1.gthr, (size_t)ctx->Bpad_max * (2 + ctx->num_sms / 2));
        CK(cudaMemsetAsync(S1.qs, 0, (size_t)ctx->Bpad_max * ds * 2, s));
        st = encode_map(ctx, &S1.tm_q, S1.qs, (uint64_t)ctx->Bpad_max, (uint64_t)ds, kTileM);
        if (st != RB_OK) return st;
        ALLOC(S1.q32, mb * d);
      }
      int lo = 0, hi = 0;
      CK(cudaDeviceGetStreamPriorityRange(&lo, &hi));   // lo = least priority
      CK(cudaStreamCreateWithPriority(&ctx->front, cudaStreamNonBlocking, lo));
      CK(cudaStreamCreateWithPriority(&ctx->front2, cudaStreamNonBlocking, lo));
      CK(cudaStreamCreateWithPriority(&ctx->sstage, cudaStreamNonBlocking, hi));
      CK(cudaEventCreateWithFlags(&ctx->ev_bigfin, cudaEventDisableTiming));
      for (int j = 0; j < kSlots; ++j) {
        CK(cudaEventCreateWithFlags(&ctx->slot[j].ev_stage, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->slot[j].ev_front, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->slot[j].ev_back, cudaEventDisableTiming));
      }
      // pinned blocks of the asynchronous host path
      ctx->az_off_plen = ((size_t)kTileM * d * 4 + 255) & ~(size_t)255;
      ctx->az_off_assign = ctx->az_off_plen + 512;
      ctx->az_off_flag = ctx->az_off_assign + 512;
      for (int j = 0; j < kSlots; ++j) {
        rb_ctx::AsyncSlot& A = ctx->async[j];
        if (cudaHostAlloc((void**)&A.h, ctx->az_off_flag + 256, cudaHostAllocMapped) != cudaSuccess ||
            cudaHostGetDevicePointer((void**)&A.d, A.h, 0) != cudaSuccess) {
          cudaGetLastError();
          if (A.h) cudaFreeHost(A.h);
          A.h = A.d = nullptr;   // no mapped pinned memory: rb_decide_submit returns RB_EUNSUPPORTED
        } else {
          std::memset(A.h, 0, ctx->az_off_flag + 256);
        }
      }
    }
    CK(scan_tc_prepare());
    CK(scan_tc2_prepare());
  }
  {
    rb_ctx::Slot& S0 = ctx->slot[0];   // the primary buffer set
    S0.qs = ctx->qs; S0.tm_q = ctx->tm_q; S0.part_sim = ctx->part_sim; S0.part_idx = ctx->part_idx; S0.q32 = ctx->q32;
    S0.gthr = ctx->gthr;
    S0.pred_q = ctx->pred_q; S0.pred_l = ctx->pred_l; S0.termA = ctx->termA; S0.termP = ctx->termP; S0.key = ctx->key;
  }
  {
    const int rr = opt.rerank_slack > 0 ? 1 : 0;
    const size_t fin = std::max({finish_smem_bytes(ctx->num_sms * scan_tc_replicas(1, ctx->ks, ctx->num_sms), ctx->ks, ctx->kc, d, rr),
                                 finish_smem_bytes(ctx->num_sms / 2 + 1, ctx->kcap, ctx->kc, d, rr),
                                 finish_smem_bytes(1, ctx->kc, ctx->kc, d, rr)});
    CK(finish_prepare(fin));
    CK(lpt_dispatch_prepare());
  }
  ALLOC(ctx->scratch_nn_idx, mb * k);
  ALLOC(ctx->scratch_nn_sim, mb * k);
#undef ALLOC
  CK(cudaStreamSynchronize(s));   // the caller may free its buffers on return
  return RB_OK;
}

rb_status rb_set_instances(rb_ctx* ctx, int32_t I, const int32_t* tier, const int32_t* cap, const float* price_in,
                           const float* price_out, const rb_lat_head* heads) {
  if (!ctx) return RB_EINVAL;
  if (!tier || !cap || !price_in || !price_out || !heads) return fail(ctx, RB_EINVAL, "NULL argument");
  if (I < 1 || I > kMaxI) return fail(ctx, RB_EINVAL, "I out of range [1,1024]");
  const int M = ctx->M;
  int32_t present[kMaxM] = {0};
  for (int i = 0; i < I; ++i) {
    if (tier[i] < 0 || tier[i] >= M) return fail(ctx, RB_EINVAL, "tier out of range");
    if (cap[i] < 1) return fail(ctx, RB_EINVAL, "cap must be >= 1");
    present[tier[i]] = 1;
  }
  float pre[kMaxM], dec[kMaxM], slope[kMaxM];
  for (int m = 0; m < M; ++m) {
    if (!finite_nonneg(price_in[m]) || !finite_nonneg(price_out[m])) return fail(ctx, RB_EINVAL, "prices must be finite, >= 0");
    if (!finite_nonneg(heads[m].prefill_ms_per_tok) || !finite_nonneg(heads[m].decode_ms_per_tok) ||
        !finite_nonneg(heads[m].batch_slope))
      return fail(ctx, RB_EINVAL, "latency head coefficients must be finite, >= 0");
    pre[m] = heads[m].prefill_ms_per_tok; dec[m] = heads[m].decode_ms_per_tok; slope[m] = heads[m].batch_slope;
  }
  std::vector<float> dec_i(I), slope_i(I);
  for (int i = 0; i < I; ++i) { dec_i[i] = dec[tier[i]]; slope_i[i] = slope[tier[i]]; }
  std::vector<int32_t> members, tstart(kMaxM + 1, 0);   // pipeline mode: instances by (tier, index)
  for (int m = 0; m < M; ++m) {
    tstart[m] = (int32_t)members.size();
    for (int i = 0; i < I; ++i)
      if (tier[i] == m) members.push_back(i);
  }
  for (int m = M; m <= kMaxM; ++m) tstart[m] = (int32_t)members.size();
  cudaStream_t s = ctx->stream;
  // scores buffers depend on I
  if (I != ctx->I) {
    CK(cudaStreamSynchronize(s));
    cudaFree(ctx->scores); cudaFree(ctx->scores0);
    ctx->scores = ctx->scores0 = nullptr;
    const size_t n = (size_t)ctx->opt.max_batch * I;
    if (dev_alloc(&ctx->scores, n) != cudaSuccess || dev_alloc(&ctx->scores0, n) != cudaSuccess) {
      cudaGetLastError();
      ctx->I = 0;
      return fail(ctx, RB_ENOMEM, "cudaMalloc scores");
    }
    drop_graphs(ctx);   // grid shapes depend on I
  }
  CK(cudaMemcpyAsync(ctx->tier, tier, I * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->cap, cap, I * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->present, present, M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->price_in, price_in, M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->price_out, price_out, M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->pre, pre, M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->dec, dec, M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->slope, slope, M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->dec_i, dec_i.data(), I * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->slope_i, slope_i.data(), I * 4, cudaMemcpyHostToDevice, s));
  ctx->n_pending = 0;   // the state is reset
  CK(cudaMemcpyAsync(ctx->members, members.data(), I * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->tstart, tstart.data(), (kMaxM + 1) * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemsetAsync(ctx->pipe_cursor, 0, kMaxM * 4, s));
  CK(cudaMemsetAsync(ctx->pipe_counter, 0, 8, s));
  CK(cudaMemsetAsync(ctx->dq, 0, kMaxI * 4, s));
  CK(cudaMemsetAsync(ctx->bq, 0, kMaxI * 4, s));
  CK(cudaMemsetAsync(ctx->f_aux, 0, (size_t)kMaxI * kMaxFeatures * 4, s));
  CK(cudaStreamSynchronize(s));   // stack arrays above are read by pageable copies
  ctx->I = I;
  return RB_OK;
}

rb_status rb_set_tpot_forest(rb_ctx* ctx, const rb_tree_node* nodes, int32_t n_nodes, const int32_t* tree_root,
                             int32_t n_trees, const int32_t* tier_tree_begin, const float* base, int32_t n_features) {
  if (!ctx) return RB_EINVAL;
  if (!nodes || !tree_root || !tier_tree_begin || !base) return fail(ctx, RB_EINVAL, "NULL argument");
  if (n_nodes < 1 || n_nodes > (1 << 22) || n_trees < 0) return fail(ctx, RB_EINVAL, "forest size out of range");
  if (n_features < 2 || n_features > kMaxFeatures) return fail(ctx, RB_EINVAL, "n_features out of range [2,8]");
  const int M = ctx->M;
  if (tier_tree_begin[0] != 0 || tier_tree_begin[M] != n_trees) return fail(ctx, RB_EINVAL, "tier_tree_begin must span [0,n_trees]");
  for (int m = 0; m < M; ++m) {
    const int n = tier_tree_begin[m + 1] - tier_tree_begin[m];
    if (n < 0 || n > kMaxTreesPerTier) return fail(ctx, RB_EINVAL, "trees per tier out of range [0,256]");
    if (!std::isfinite(base[m])) return fail(ctx, RB_EINVAL, "base must be finite");
  }
  for (int j = 0; j < n_trees; ++j)
    if (tree_root[j] < 0 || tree_root[j] >= n_nodes) return fail(ctx, RB_EINVAL, "tree_root out of range");
  for (int n = 0; n < n_nodes; ++n) {
    if (!std::isfinite(nodes[n].value)) return fail(ctx, RB_EINVAL, "node value must be finite");
    if (nodes[n].feature < 0) continue;
    if (nodes[n].feature >= n_features) return fail(ctx, RB_EINVAL, "node feature out of range");
    // children after their parent: every walk is finite
    if (nodes[n].left <= n || nodes[n].left >= n_nodes || nodes[n].right <= n || nodes[n].right >= n_nodes)
      return fail(ctx, RB_EINVAL, "node children must lie after their parent and inside the node array");
  }
  // The nodes are stored tier by tier (each tree copied out in pre-order, child links re-pointed): the dispatch kernel
  // keeps the nodes of the tier it is evaluating in shared memory (a walk is then a chain of shared-memory reads, not of
  // L2 round trips).  Pure re-arrangement of the caller's forest: every walk visits the same tests and the same leaf.
  std::vector<rb_tree_node> pk;
  std::vector<int32_t> root2((size_t)n_trees), nbegin((size_t)M + 1, 0);
  pk.reserve((size_t)n_nodes);
  int max_tier_nodes = 0;
  double tpot_hi = 1e-6;   // |base| + sum over the tier's trees of the largest |leaf|: no evaluation exceeds it
  for (int m = 0; m < M; ++m) {
    nbegin[m] = (int32_t)pk.size();
    double tier_hi = std::fabs((double)base[m]);
    for (int tr = tier_tree_begin[m]; tr < tier_tree_begin[m + 1]; ++tr) {
      double leaf_hi = 0.0;
      std::vector<std::pair<int32_t, int32_t>> todo;   // (old node, slot of the link to patch; -1: the root)
      todo.push_back({tree_root[tr], -1});
      while (!todo.empty()) {
        const auto [old, link] = todo.back();
        todo.pop_back();
        const int32_t id = (int32_t)pk.size();
        if (pk.size() >= ((size_t)1 << 23)) return fail(ctx, RB_EINVAL, "forest too large once its trees are unshared");
        pk.push_back(nodes[old]);
        if (link < 0) root2[tr] = id;
        else if (link & 1) pk[link >> 1].right = id;
        else pk[link >> 1].left = id;
        if (nodes[old].feature >= 0) {
          todo.push_back({nodes[old].right, 2 * id + 1});
          todo.push_back({nodes[old].left, 2 * id});
        } else {
          leaf_hi = std::max(leaf_hi, std::fabs((double)nodes[old].value));
        }
      }
      tier_hi += leaf_hi;
    }
    tpot_hi = std::max(tpot_hi, tier_hi);
    max_tier_nodes = std::max(max_tier_nodes, (int)pk.size() - nbegin[m]);
  }
  nbegin[M] = (int32_t)pk.size();
  // The packed copy for the dispatch loop's shared-memory cache (ForestDev::cwords): 8 bytes per inner node, 4 per leaf,
  // so that a whole forest of the paper's size class stays resident (64 trees of depth 5 per tier, 8 tiers: 190 KB
  // against 516 KB of 16-byte nodes).  Same tests, same leaves: a re-encoding.
  std::vector<uint32_t> cw;
  std::vector<int32_t> cbegin((size_t)M + 1, 0);
  int max_tier_cwords = 0;
  {
    auto bits = [](float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; };
    std::vector<uint32_t> off(pk.size(), 0);
    for (int m = 0; m < M; ++m) {
      cbegin[m] = (int32_t)cw.size();
      const int t0 = tier_tree_begin[m], t1 = tier_tree_begin[m + 1];
      uint32_t o = (uint32_t)(t1 - t0);   // the roots come first
      for (int n = nbegin[m]; n < nbegin[m + 1]; ++n) {   // pre-order: offsets in node order
        off[n] = o;
        o += pk[n].feature >= 0 ? 2u : 1u;
      }
      if (o >= (1u << 27)) return fail(ctx, RB_EINVAL, "forest too large for the packed encoding");
      cw.resize((size_t)cbegin[m] + o, 0u);
      uint32_t* blk = cw.data() + cbegin[m];
      for (int tr = t0; tr < t1; ++tr) blk[tr - t0] = (off[root2[tr]] << 1) | (pk[root2[tr]].feature < 0 ? 1u : 0u);
      for (int n = nbegin[m]; n < nbegin[m + 1]; ++n) {
        if (pk[n].feature < 0) {
          blk[off[n]] = bits(pk[n].value);
        } else {
          const int l = pk[n].left, r = pk[n].right;   // l == n + 1 (pre-order)
          blk[off[n]] = bits(pk[n].value);
          blk[off[n] + 1] = (uint32_t)pk[n].feature | (pk[l].feature < 0 ? 8u : 0u) | (pk[r].feature < 0 ? 16u : 0u) |
                            ((off[r] - off[n]) << 5);
        }
      }
      max_tier_cwords = std::max(max_tier_cwords, (int)o);
    }
    cbegin[M] = (int32_t)cw.size();
  }
  cudaStream_t s = ctx->stream;
  CK(cudaStreamSynchronize(s));
  cudaFree(ctx->f_nodes); cudaFree(ctx->f_root); cudaFree(ctx->f_begin); cudaFree(ctx->f_base); cudaFree(ctx->f_nbegin);
  cudaFree(ctx->f_cwords); cudaFree(ctx->f_cbegin);
  ctx->f_nodes = nullptr; ctx->f_root = ctx->f_begin = ctx->f_nbegin = nullptr; ctx->f_base = nullptr;
  ctx->f_cwords = nullptr; ctx->f_cbegin = nullptr;
  ctx->f_total_cwords = (int)cw.size(); ctx->f_max_tier_cwords = max_tier_cwords;
  ctx->f_max_tier_nodes = max_tier_nodes;
  ctx->f_tpot_hi = (float)std::min(2.0 * tpot_hi, 3.0e38);   // (doubled: the fp32 sum rounds)
  ctx->has_forest = false;
  static_assert(sizeof(rb_tree_node) == sizeof(int4), "rb_tree_node is read as int4");
  if (dev_alloc(&ctx->f_nodes, pk.size()) != cudaSuccess || dev_alloc(&ctx->f_root, (size_t)n_trees) != cudaSuccess ||
      dev_alloc(&ctx->f_begin, (size_t)M + 1) != cudaSuccess || dev_alloc(&ctx->f_base, (size_t)M) != cudaSuccess ||
      dev_alloc(&ctx->f_nbegin, (size_t)M + 1) != cudaSuccess || dev_alloc(&ctx->f_cwords, cw.size()) != cudaSuccess ||
      dev_alloc(&ctx->f_cbegin, (size_t)M + 1) != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, RB_ENOMEM, "cudaMalloc forest");
  }
  CK(cudaMemcpyAsync(ctx->f_nodes, pk.data(), pk.size() * sizeof(rb_tree_node), cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->f_root, root2.data(), (size_t)n_trees * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->f_begin, tier_tree_begin, (size_t)(M + 1) * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->f_nbegin, nbegin.data(), (size_t)(M + 1) * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->f_base, base, (size_t)M * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->f_cwords, cw.data(), cw.size() * 4, cudaMemcpyHostToDevice, s));
  CK(cudaMemcpyAsync(ctx->f_cbegin, cbegin.data(), (size_t)(M + 1) * 4, cudaMemcpyHostToDevice, s));
  CK(cudaStreamSynchronize(s));
  if (n_features != ctx->f_features) CK(cudaMemsetAsync(ctx->f_aux, 0, (size_t)kMaxI * kMaxFeatures * 4, s));
  ctx->f_features = n_features;
  ctx->has_forest = true;
  drop_graphs(ctx);   // captured kernel arguments hold the old forest
  return RB_OK;
}

rb_status rb_set_telemetry(rb_ctx* ctx, const float* aux) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_set_telemetry before rb_set_instances");
  if (!ctx->has_forest) return fail(ctx, RB_ESTATE, "rb_set_telemetry before rb_set_tpot_forest");
  const int Fa = ctx->f_features - 2;
  if (Fa == 0) return RB_OK;
  if (!aux) return fail(ctx, RB_EINVAL, "NULL argument");
  CK(cudaMemcpyAsync(ctx->f_aux, aux, (size_t)ctx->I * Fa * 4, cudaMemcpyDefault, ctx->stream));
  if (is_host_ptr(aux)) CK(cudaStreamSynchronize(ctx->stream));
  return RB_OK;
}

rb_status rb_set_state(rb_ctx* ctx, const float* queued_tokens, const int32_t* running) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_set_state before rb_set_instances");
  if (!queued_tokens || !running) return fail(ctx, RB_EINVAL, "NULL argument");
  const bool host = is_host_ptr(queued_tokens) || is_host_ptr(running);
  if (is_host_ptr(queued_tokens) && is_host_ptr(running)) {
    for (int i = 0; i < ctx->I; ++i)
      if (!finite_nonneg(queued_tokens[i]) || running[i] < 0) return fail(ctx, RB_EINVAL, "state must be finite, >= 0");
  }
  ctx->n_pending = 0;   // advances before an overwrite of the whole state have no effect
  CK(cudaMemcpyAsync(ctx->dq, queued_tokens, ctx->I * 4, cudaMemcpyDefault, ctx->stream));
  CK(cudaMemcpyAsync(ctx->bq, running, ctx->I * 4, cudaMemcpyDefault, ctx->stream));
  if (host) CK(cudaStreamSynchronize(ctx->stream));
  return RB_OK;
}

rb_status rb_get_state(rb_ctx* ctx, float* queued_tokens, int32_t* running) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_get_state before rb_set_instances");
  {
    rb_status st = flush_pending(ctx);
    if (st != RB_OK) return st;
  }
  bool any_host = false;
  if (queued_tokens) {
    any_host |= is_host_ptr(queued_tokens);
    CK(cudaMemcpyAsync(queued_tokens, ctx->dq, ctx->I * 4, cudaMemcpyDefault, ctx->stream));
  }
  if (running) {
    any_host |= is_host_ptr(running);
    CK(cudaMemcpyAsync(running, ctx->bq, ctx->I * 4, cudaMemcpyDefault, ctx->stream));
  }
  if (any_host) CK(cudaStreamSynchronize(ctx->stream));
  return RB_OK;
}

rb_status rb_advance_state(rb_ctx* ctx, float elapsed_ms) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_advance_state before rb_set_instances");
  if (!finite_nonneg(elapsed_ms)) return fail(ctx, RB_EINVAL, "elapsed_ms must be finite and >= 0");
  if (ctx->opt.latency_mode == 2) {
    if (!ctx->has_forest) return fail(ctx, RB_ESTATE, "latency_mode 2 needs rb_set_tpot_forest first");
    CK(launch_tpot_forest(table_of(ctx), forest_of(ctx), ctx->dq, ctx->bq, nullptr, elapsed_ms, ctx->stream));
  } else {
    // deferred: the next rb_decide applies it in its first kernel (one launch less per decision); any other reader or
    // writer of the state applies it first (flush_pending)
    if (ctx->n_pending == kMaxPendingAdvance) {
      rb_status st = flush_pending(ctx);
      if (st != RB_OK) return st;
    }
    ctx->pending_adv[ctx->n_pending++] = elapsed_ms;
    return RB_OK;
  }
  ctx->launches += 1;
  return RB_OK;
}

rb_status rb_batch_target(rb_ctx* ctx, int32_t bs_min, int32_t bs_max, int32_t* target, int32_t* n_busy) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_batch_target before rb_set_instances");
  if (!target) return fail(ctx, RB_EINVAL, "NULL argument");
  if (bs_min < 1 || bs_max < bs_min) return fail(ctx, RB_EINVAL, "need 1 <= bs_min <= bs_max");
  rb_status st = flush_pending(ctx);   // the rule reads the current state
  if (st != RB_OK) return st;
  const bool h_t = is_host_ptr(target), h_b = n_busy && is_host_ptr(n_busy);
  int32_t* d_out = ctx->order;   // two words of per-decision scratch (free between decisions)
  int32_t* d_t = h_t ? d_out : target;
  int32_t* d_b = n_busy ? (h_b ? d_out + 1 : n_busy) : nullptr;
  CK(launch_batch_target(table_of(ctx), ctx->bq, bs_min, bs_max, d_t, d_b, ctx->stream));
  ctx->launches += 1;
  if (h_t) CK(cudaMemcpyAsync(target, d_t, 4, cudaMemcpyDeviceToHost, ctx->stream));
  if (h_b) CK(cudaMemcpyAsync(n_busy, d_b, 4, cudaMemcpyDeviceToHost, ctx->stream));
  if (h_t || h_b) CK(cudaStreamSynchronize(ctx->stream));
  return RB_OK;
}

rb_status rb_decide(rb_ctx* ctx, const float* query_emb, const int32_t* prompt_len, int32_t B, const float w[3],
                    int32_t* assignment, float* scores, float* pred_quality, float* pred_outlen, int32_t* nn_idx,
                    float* nn_sim) {
  return rb_decide_budgeted(ctx, query_emb, prompt_len, nullptr, B, w, assignment, nullptr, scores, pred_quality,
                            pred_outlen, nn_idx, nn_sim);
}

rb_status rb_decide_budgeted(rb_ctx* ctx, const float* query_emb, const int32_t* prompt_len, const float* budget,
                             int32_t B, const float w[3], int32_t* assignment, int32_t* max_tokens, float* scores,
                             float* pred_quality, float* pred_outlen, int32_t* nn_idx, float* nn_sim) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_decide before rb_set_instances");
  if (ctx->opt.latency_mode == 2 && !ctx->has_forest) return fail(ctx, RB_ESTATE, "latency_mode 2 needs rb_set_tpot_forest first");
  if (!query_emb || !prompt_len || !assignment) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > ctx->opt.max_batch) return fail(ctx, RB_EINVAL, "B out of range [1,max_batch]");
  rb_status st = check_weights(ctx, w);
  if (st != RB_OK) return st;
  const size_t bm = (size_t)B * ctx->M * 4, bk = (size_t)B * ctx->k * 4;
  Stager sg{ctx};
  CallParams cp{};
  cp.w_qual = w[0]; cp.w_lat = w[1]; cp.w_cost = w[2]; cp.commit = 1;
  bool adv_folded = false;
  if (ctx->opt.latency_mode != 2) {
    cp.n_adv = ctx->n_pending;   // applied by the dispatch kernel when it loads the state
    for (int a = 0; a < ctx->n_pending; ++a) cp.adv_ms[a] = ctx->pending_adv[a];
    adv_folded = true;           // (n_pending is cleared only once the decision has been enqueued: a failed call changes nothing)
  } else {
    st = flush_pending(ctx);
    if (st != RB_OK) return st;
  }
  // (the fp32-storage scan reads every query from every block: it wants them in device memory)
  // (host queries: read in place from the pinned block by the staging kernel, which -- under fp32 storage -- also leaves
  // the device copy the re-rank reads; the copy-engine fallback stages them in a separate buffer)
  cp.query = sg.in_zc(query_emb, 0, ctx->zc_query_cap, ctx->q32_in, (size_t)B * ctx->d * 4);
  cp.plen = sg.in_zc(prompt_len, ctx->zc_off_plen, (size_t)B * 4, ctx->plen, (size_t)B * 4);
  cp.q_src = ctx->pred_q;
  cp.l_src = ctx->pred_l;
  cp.budget = budget ? sg.in_zc(budget, ctx->zc_off_budget, (size_t)B * 4, ctx->budget, (size_t)B * 4) : nullptr;
  // (with max_tokens the dispatch kernel reads the assignment back: it then stays in device memory)
  cp.assignment = max_tokens ? sg.out(assignment, ctx->assignment, (size_t)B * 4)
                             : sg.out_zc(assignment, ctx->zc_off_assign, ctx->assignment, (size_t)B * 4);
  cp.max_tokens = sg.out(max_tokens, ctx->max_tokens, (size_t)B * 4);
  cp.scores = sg.out(scores, ctx->scores, (size_t)B * ctx->I * 4);
  cp.pred_q = sg.out_internal(pred_quality, ctx->pred_q, bm);
  cp.pred_l = sg.out_internal(pred_outlen, ctx->pred_l, bm);
  cp.nn_idx = sg.out(nn_idx, ctx->scratch_nn_idx, bk);
  cp.nn_sim = sg.out(nn_sim, ctx->scratch_nn_sim, bk);
  if (sg.err != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaMemcpyAsync (inputs)", sg.err);
  if (sg.wait_flag && !sg.needs_sync && !ctx->stage_timing) {
    cp.done_flag = reinterpret_cast<uint32_t*>(ctx->d_zc + ctx->zc_off_flag);
    cp.done_seq = ++ctx->done_seq;
  } else {
    sg.needs_sync = sg.any_host;
  }
  // throughput mode: device buffers only (host buffers make the call synchronous anyway)
  const bool pipelined = ctx->front != nullptr && !sg.any_host && adv_folded && !ctx->stage_timing &&
                         ctx->opt.use_graph != 0;
  if (pipelined) {
    const rb_ctx::Slot& S = ctx->slot[ctx->pipe_seq % kSlots];
    cp.q_src = S.pred_q;
    cp.l_src = S.pred_l;
  }
  st = push_params(ctx, cp);
  if (st != RB_OK) return st;
  st = pipelined ? run_pipelined(ctx, B) : run_path(ctx, B, 0);
  if (st != RB_OK) return st;
  if (adv_folded) ctx->n_pending = 0;
  collect_stage_times(ctx, 0);
  return sg.finish();
}

rb_status rb_decide_submit(rb_ctx* ctx, const float* query_emb, const int32_t* prompt_len, int32_t B, const float w[3]) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_decide_submit before rb_set_instances");
  if (!ctx->front) return fail(ctx, RB_ESTATE, "rb_decide_submit needs rb_options.pipeline = 1");
  if (ctx->opt.latency_mode == 2 || !ctx->opt.use_graph || ctx->stage_timing)
    return fail(ctx, RB_EUNSUPPORTED, "rb_decide_submit: linear or static latency head, graph replay on, stage timing off");
  if (!query_emb || !prompt_len) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > kTileM || B > ctx->opt.max_batch) return fail(ctx, RB_EINVAL, "B out of range [1, min(128, max_batch)]");
  rb_status st = check_weights(ctx, w);
  if (st != RB_OK) return st;
  if (ctx->async_tail - ctx->async_head >= (uint64_t)kSlots)
    return fail(ctx, RB_ESTATE, "three decisions in flight: rb_decide_collect first");
  // the buffer set the next pipelined decision uses decides the pinned block
  rb_ctx::AsyncSlot& A = ctx->async[ctx->pipe_seq % kSlots];
  if (!A.h) return fail(ctx, RB_EUNSUPPORTED, "no mapped pinned host memory");
  if (A.busy) return fail(ctx, RB_ESTATE, "the buffer set of this submission is still in flight: rb_decide_collect first");
  std::memcpy(A.h, query_emb, (size_t)B * ctx->d * 4);
  std::memcpy(A.h + ctx->az_off_plen, prompt_len, (size_t)B * 4);
  CallParams cp{};
  cp.w_qual = w[0]; cp.w_lat = w[1]; cp.w_cost = w[2]; cp.commit = 1;
  cp.n_adv = ctx->n_pending;
  for (int a = 0; a < ctx->n_pending; ++a) cp.adv_ms[a] = ctx->pending_adv[a];
  cp.query = reinterpret_cast<const float*>(A.d);
  cp.plen = reinterpret_cast<const int32_t*>(A.d + ctx->az_off_plen);
  cp.assignment = reinterpret_cast<int32_t*>(A.d + ctx->az_off_assign);
  cp.done_flag = reinterpret_cast<uint32_t*>(A.d + ctx->az_off_flag);
  cp.done_seq = ++ctx->done_seq;
  const rb_ctx::Slot& S = ctx->slot[ctx->pipe_seq % kSlots];
  cp.q_src = S.pred_q;
  cp.l_src = S.pred_l;
  st = push_params(ctx, cp);
  if (st != RB_OK) return st;
  st = run_pipelined(ctx, B);
  if (st != RB_OK) return st;
  ctx->n_pending = 0;
  A.busy = true;
  A.seq = cp.done_seq;
  A.B = B;
  ctx->async_tail += 1;
  return RB_OK;
}

rb_status rb_decide_collect(rb_ctx* ctx, int32_t* assignment, int32_t B) {
  if (!ctx) return RB_EINVAL;
  if (!assignment) return fail(ctx, RB_EINVAL, "NULL argument");
  if (ctx->async_tail == ctx->async_head) return fail(ctx, RB_ESTATE, "rb_decide_collect: nothing in flight");
  // submissions rotate through the blocks in submission order, unless synchronous pipelined calls came in
  // between: the oldest one in flight is the busy block with the smaller sequence number
  rb_ctx::AsyncSlot* A = nullptr;
  for (auto& c : ctx->async)
    if (c.busy && (!A || (int32_t)(c.seq - A->seq) < 0)) A = &c;
  if (!A) return fail(ctx, RB_ESTATE, "rb_decide_collect: nothing in flight");
  if (B != A->B) return fail(ctx, RB_EINVAL, "rb_decide_collect: B differs from the submitted batch");
  volatile uint32_t* flag = reinterpret_cast<volatile uint32_t*>(A->h + ctx->az_off_flag);
  for (uint32_t spins = 1; *flag != A->seq; ++spins) {
    if ((spins & 0x3fff) == 0) {
      const cudaError_t q = cudaStreamQuery(ctx->stream);
      if (q == cudaSuccess) break;
      if (q != cudaErrorNotReady) return fail(ctx, RB_ECUDA, "cudaStreamQuery", q);
    }
  }
  if (*flag != A->seq) CK(cudaStreamSynchronize(ctx->stream));
  std::memcpy(assignment, A->h + ctx->az_off_assign, (size_t)B * 4);
  A->busy = false;
  ctx->async_head += 1;
  return RB_OK;
}

rb_status rb_estimate(rb_ctx* ctx, const float* query_emb, int32_t B, float* pred_quality, float* pred_outlen,
                      int32_t* nn_idx, float* nn_sim) {
  if (!ctx) return RB_EINVAL;
  if (!query_emb) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > ctx->opt.max_batch) return fail(ctx, RB_EINVAL, "B out of range [1,max_batch]");
  const size_t bm = (size_t)B * ctx->M * 4, bk = (size_t)B * ctx->k * 4;
  Stager sg{ctx};
  CallParams cp{};
  cp.query = sg.in(query_emb, ctx->q32_in, (size_t)B * ctx->d * 4);
  cp.pred_q = sg.out_internal(pred_quality, ctx->pred_q, bm);
  cp.pred_l = sg.out_internal(pred_outlen, ctx->pred_l, bm);
  cp.nn_idx = sg.out(nn_idx, ctx->scratch_nn_idx, bk);
  cp.nn_sim = sg.out(nn_sim, ctx->scratch_nn_sim, bk);
  if (sg.err != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaMemcpyAsync (inputs)", sg.err);
  rb_status st = push_params(ctx, cp);
  if (st != RB_OK) return st;
  st = run_path(ctx, B, 1);
  if (st != RB_OK) return st;
  collect_stage_times(ctx, 1);
  return sg.finish();
}

rb_status rb_decide_from_predictions(rb_ctx* ctx, const float* quality, const float* outlen, const int32_t* prompt_len,
                                     int32_t B, const float w[3], int32_t commit, int32_t* assignment, float* scores,
                                     float* scores0, int32_t* order) {
  return rb_decide_from_predictions_budgeted(ctx, quality, outlen, prompt_len, nullptr, B, w, commit, assignment, nullptr,
                                             scores, scores0, order);
}

rb_status rb_decide_from_predictions_budgeted(rb_ctx* ctx, const float* quality, const float* outlen,
                                              const int32_t* prompt_len, const float* budget, int32_t B, const float w[3],
                                              int32_t commit, int32_t* assignment, int32_t* max_tokens, float* scores,
                                              float* scores0, int32_t* order) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_decide_from_predictions before rb_set_instances");
  if (ctx->opt.latency_mode == 2 && !ctx->has_forest) return fail(ctx, RB_ESTATE, "latency_mode 2 needs rb_set_tpot_forest first");
  if (!quality || !outlen || !prompt_len || !assignment) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > ctx->opt.max_batch) return fail(ctx, RB_EINVAL, "B out of range [1,max_batch]");
  rb_status st = check_weights(ctx, w);
  if (st != RB_OK) return st;
  const size_t bm = (size_t)B * ctx->M * 4, bi = (size_t)B * ctx->I * 4;
  Stager sg{ctx};
  CallParams cp{};
  cp.w_qual = w[0]; cp.w_lat = w[1]; cp.w_cost = w[2]; cp.commit = commit ? 1 : 0;
  st = flush_pending(ctx);   // the score kernel's CTAs all read the state: it must be current before they start
  if (st != RB_OK) return st;
  cp.q_src = sg.in(quality, ctx->stage_q, bm);
  cp.l_src = sg.in(outlen, ctx->stage_l, bm);
  cp.plen = sg.in(prompt_len, ctx->plen, (size_t)B * 4);
  cp.budget = budget ? sg.in(budget, ctx->budget, (size_t)B * 4) : nullptr;
  cp.assignment = sg.out(assignment, ctx->assignment, (size_t)B * 4);
  cp.max_tokens = sg.out(max_tokens, ctx->max_tokens, (size_t)B * 4);
  cp.scores = sg.out(scores, ctx->scores, bi);
  cp.scores0 = sg.out(scores0, ctx->scores0, bi);
  cp.order = sg.out(order, ctx->order, (size_t)B * 4);
  if (sg.err != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaMemcpyAsync (inputs)", sg.err);
  st = push_params(ctx, cp);
  if (st != RB_OK) return st;
  st = run_path(ctx, B, 2);
  if (st != RB_OK) return st;
  collect_stage_times(ctx, 2);
  return sg.finish();
}

rb_status rb_decide_from_predictions_static(rb_ctx* ctx, const float* quality, const float* outlen,
                                            const int32_t* prompt_len, int32_t B, const float w[3], int32_t commit,
                                            int32_t* assignment) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_decide_from_predictions_static before rb_set_instances");
  if (ctx->opt.latency_mode == 2 && !ctx->has_forest) return fail(ctx, RB_ESTATE, "latency_mode 2 needs rb_set_tpot_forest first");
  if (!quality || !outlen || !prompt_len || !assignment) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > static_scratch_max_b() || (long long)B * ctx->M > static_scratch_max_bm()) {
    char buf[160];
    snprintf(buf, sizeof buf, "rb_decide_from_predictions_static: B = %d with M = %d exceeds the static scratch (1 <= B <= %d and B * M <= %d)",
             (int)B, ctx->M, static_scratch_max_b(), static_scratch_max_bm());
    return fail(ctx, RB_EINVAL, buf);
  }
  // (host buffers would need staging copies through allocated memory and a stream synchronisation: not this entry point)
  if (is_host_ptr(quality) || is_host_ptr(outlen) || is_host_ptr(prompt_len) || is_host_ptr(assignment))
    return fail(ctx, RB_EINVAL, "rb_decide_from_predictions_static: quality, outlen, prompt_len and assignment must be device memory");
  rb_status st = check_weights(ctx, w);
  if (st != RB_OK) return st;
  st = flush_pending(ctx);   // the score kernel's CTAs all read the state: it must be current before they start
  if (st != RB_OK) return st;
  CallParams cp{};
  cp.w_qual = w[0]; cp.w_lat = w[1]; cp.w_cost = w[2]; cp.commit = commit ? 1 : 0;
  cp.q_src = quality;
  cp.l_src = outlen;
  cp.plen = prompt_len;
  cp.assignment = assignment;
  InstTable t = table_of(ctx);
  if (ctx->opt.latency_mode == 2) {   // the head over the batch-start state
    CK(launch_tpot_forest(t, forest_of(ctx), ctx->dq, ctx->bq, ctx->f_tpot0, -1.0f, ctx->stream));
    ctx->launches += 1;
  }
  CK(launch_score_dispatch_static(t, ctx->dq, ctx->bq, cp, B, modes_of(ctx), forest_of(ctx), ctx->stream));
  ctx->launches += 2;
  return RB_OK;
}

rb_status rb_sweep_weights(rb_ctx* ctx, const float* quality, const float* outlen, const int32_t* prompt_len,
                           const float* budget, int32_t B, const float* w, int32_t P, int32_t* assignment) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_sweep_weights before rb_set_instances");
  if (ctx->opt.latency_mode == 2 && !ctx->has_forest) return fail(ctx, RB_ESTATE, "latency_mode 2 needs rb_set_tpot_forest first");
  if (!quality || !outlen || !prompt_len || !w || !assignment) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > ctx->opt.max_batch) return fail(ctx, RB_EINVAL, "B out of range [1,max_batch]");
  if (P < 1 || P > 65535) return fail(ctx, RB_EINVAL, "P out of range [1,65535]");
  if (is_host_ptr(w) == false) return fail(ctx, RB_EINVAL, "w must be host memory");
  rb_status st = RB_OK;
  for (int p = 0; p < P; ++p)
    if ((st = check_weights(ctx, w + 3 * p)) != RB_OK) return st;
  st = flush_pending(ctx);
  if (st != RB_OK) return st;
  // per-point scratch, grown on demand
  const size_t pb = (size_t)P * B, pbm = pb * ctx->M;
  auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
  const size_t o_w = 0, o_a = al((size_t)P * 12), o_p = o_a + al(pbm * 4), o_k = o_p + al(pbm * 4), o_asg = o_k + al(pb * 4),
               need = o_asg + al(pb * 4);
  if (need > ctx->sweep_cap) {
    CK(cudaStreamSynchronize(ctx->stream));
    if (ctx->sweep_buf) cudaFree(ctx->sweep_buf);
    ctx->sweep_buf = nullptr;
    ctx->sweep_cap = 0;
    cudaError_t e = cudaMalloc((void**)&ctx->sweep_buf, need);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, RB_ENOMEM, "cudaMalloc sweep scratch", e); }
    ctx->sweep_cap = need;
  }
  uint8_t* sb = ctx->sweep_buf;
  CK(cudaMemcpyAsync(sb + o_w, w, (size_t)P * 12, cudaMemcpyHostToDevice, ctx->stream));
  const size_t bm = (size_t)B * ctx->M * 4;
  Stager sg{ctx};
  CallParams cp{};
  cp.commit = 0;
  cp.q_src = sg.in(quality, ctx->stage_q, bm);
  cp.l_src = sg.in(outlen, ctx->stage_l, bm);
  cp.plen = sg.in(prompt_len, ctx->plen, (size_t)B * 4);
  cp.budget = budget ? sg.in(budget, ctx->budget, (size_t)B * 4) : nullptr;
  cp.assignment = sg.out(assignment, reinterpret_cast<int32_t*>(sb + o_asg), pb * 4);
  cp.sweep_w = reinterpret_cast<const float*>(sb + o_w);
  if (sg.err != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaMemcpyAsync (inputs)", sg.err);
  st = push_params(ctx, cp);
  if (st != RB_OK) return st;
  InstTable t = table_of(ctx);
  float* termA = reinterpret_cast<float*>(sb + o_a);
  float* termP = reinterpret_cast<float*>(sb + o_p);
  float* key = reinterpret_cast<float*>(sb + o_k);
  if (ctx->opt.latency_mode == 2) {
    CK(launch_tpot_forest(t, forest_of(ctx), ctx->dq, ctx->bq, ctx->f_tpot0, -1.0f, ctx->stream));
    ctx->launches += 1;
  }
  CK(launch_score(t, ctx->dq, ctx->bq, ctx->cp_cur, B, termA, termP, key, modes_of(ctx), forest_of(ctx), ctx->stream, P));
  CK(launch_lpt_dispatch(t, ctx->dq, ctx->bq, termA, termP, key, ctx->cp_cur, B, modes_of(ctx), forest_of(ctx), ctx->stream, P));
  ctx->launches += 2;
  return sg.finish();
}

rb_status rb_set_stage_timing(rb_ctx* ctx, int32_t enabled) {
  if (!ctx) return RB_EINVAL;
  ctx->stage_timing = enabled != 0;
  return RB_OK;
}

rb_status rb_last_stage_us(rb_ctx* ctx, float us[6]) {
  if (!ctx || !us) return RB_EINVAL;
  for (int j = 0; j < 6; ++j) us[j] = ctx->stage_us[j];
  return RB_OK;
}


rb_status rb_dispatch_pipeline(rb_ctx* ctx, const int32_t* model, const float* outlen, int32_t B, int32_t policy,
                               uint64_t seed, int32_t commit, int32_t* assignment) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_dispatch_pipeline before rb_set_instances");
  if (!model || !assignment) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > ctx->opt.max_batch) return fail(ctx, RB_EINVAL, "B out of range [1,max_batch]");
  if (policy < 0 || policy > 2) return fail(ctx, RB_EINVAL, "policy must be 0 (round-robin), 1 (shortest queue) or 2 (random)");
  rb_status st = flush_pending(ctx);
  if (st != RB_OK) return st;
  Stager sg{ctx};
  const int32_t* d_model = sg.in(model, ctx->order, (size_t)B * 4);
  const float* d_outlen = outlen ? sg.in(outlen, ctx->stage_l, (size_t)B * ctx->M * 4) : nullptr;
  int32_t* d_assign = sg.out(assignment, ctx->assignment, (size_t)B * 4);
  if (sg.err != cudaSuccess) return fail(ctx, RB_ECUDA, "cudaMemcpyAsync (inputs)", sg.err);
  CK(launch_pipeline_dispatch(table_of(ctx), ctx->members, ctx->tstart, ctx->dq, ctx->bq, d_model, d_outlen, B, policy,
                              (unsigned long long)seed, ctx->pipe_counter, ctx->pipe_cursor, commit ? 1 : 0, d_assign,
                              ctx->stream));
  ctx->launches += 1;
  return sg.finish();
}

rb_status rb_match_replay(rb_ctx* ctx, const float* scores0, int32_t B, const int32_t* quota, const int32_t* greedy,
                          int32_t* match, double* objective, int32_t* n_diverged) {
  if (!ctx) return RB_EINVAL;
  if (ctx->I == 0) return fail(ctx, RB_ESTATE, "rb_match_replay before rb_set_instances");
  if (!scores0 || !quota || !match) return fail(ctx, RB_EINVAL, "NULL argument");
  if (B < 1 || B > 4096) return fail(ctx, RB_EINVAL, "B out of range [1,4096]");
  const int I = ctx->I;
  cudaStream_t s = ctx->stream;
  // offline tool: scratch is allocated per call
  const size_t nS = (size_t)B * I * 4;
  uint8_t* scratch = nullptr;
  const size_t o_S = 0, o_q = (nS + 255) & ~(size_t)255, o_g = o_q + (((size_t)I * 4 + 255) & ~(size_t)255),
               o_m = o_g + (((size_t)B * 4 + 255) & ~(size_t)255), o_out = o_m + (((size_t)B * 4 + 255) & ~(size_t)255);
  if (cudaMalloc((void**)&scratch, o_out + 256) != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, RB_ENOMEM, "cudaMalloc (match replay scratch)");
  }
  auto done = [&](rb_status st) { cudaFree(scratch); return st; };
  const float* dS = scores0;
  const int32_t* dq = quota;
  const int32_t* dg = greedy;
  int32_t* dm = match;
  cudaError_t e = cudaSuccess;
  if (is_host_ptr(scores0)) { dS = (const float*)(scratch + o_S); e = cudaMemcpyAsync(scratch + o_S, scores0, nS, cudaMemcpyHostToDevice, s); }
  if (e == cudaSuccess && is_host_ptr(quota)) { dq = (const int32_t*)(scratch + o_q); e = cudaMemcpyAsync(scratch + o_q, quota, (size_t)I * 4, cudaMemcpyHostToDevice, s); }
  if (e == cudaSuccess && greedy && is_host_ptr(greedy)) { dg = (const int32_t*)(scratch + o_g); e = cudaMemcpyAsync(scratch + o_g, greedy, (size_t)B * 4, cudaMemcpyHostToDevice, s); }
  const bool host_match = is_host_ptr(match);
  if (host_match) dm = (int32_t*)(scratch + o_m);
  double* d_obj = (double*)(scratch + o_out);
  int32_t* d_div = (int32_t*)(scratch + o_out + 8);
  int32_t* d_status = (int32_t*)(scratch + o_out + 12);
  if (e == cudaSuccess) e = match_replay_prepare();
  if (e == cudaSuccess) e = launch_match_replay(dS, B, I, dq, dg, dm, d_obj, d_div, d_status, s);
  ctx->launches += 1;
  struct { double obj; int32_t div; int32_t status; } h{};
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, d_obj, 16, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return done(fail(ctx, RB_ECUDA, "rb_match_replay", e));
  if (h.status != 0) return done(fail(ctx, RB_EINVAL, "no feasible assignment: the quotas of the admissible instances do not cover the batch"));
  if (host_match) {
    e = cudaMemcpy(match, dm, (size_t)B * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return done(fail(ctx, RB_ECUDA, "cudaMemcpy (match)", e));
  }
  if (objective) *objective = h.obj;
  if (n_diverged) *n_diverged = greedy ? h.div : 0;
  return done(RB_OK);
}

rb_status rb_last_scan_device_us(rb_ctx* ctx, float* us) {
  if (!ctx || !us) return RB_EINVAL;
  *us = ctx->scan_device_us;
  return RB_OK;
}

rb_status rb_selftest_division(rb_ctx* ctx, uint64_t n_pairs, uint64_t seed, uint64_t* mismatches) {
  if (!ctx || !mismatches) return RB_EINVAL;
  unsigned long long* dcount = nullptr;
  CK(cudaMalloc((void**)&dcount, 8));
  cudaError_t e = cudaMemsetAsync(dcount, 0, 8, ctx->stream);
  if (e == cudaSuccess) e = launch_div_selftest(n_pairs, seed, dcount, ctx->stream);
  unsigned long long h = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, dcount, 8, cudaMemcpyDeviceToHost, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  cudaFree(dcount);
  if (e != cudaSuccess) return fail(ctx, RB_ECUDA, "rb_selftest_division", e);
  *mismatches = h;
  return RB_OK;
}

rb_status rb_testing_read_bandwidth(rb_ctx* ctx, uint64_t bytes, int32_t repeats, double* gb_per_s) {
  if (!ctx || !gb_per_s || bytes < (1u << 20) || repeats < 1) return RB_EINVAL;
  uint8_t* buf = nullptr;
  uint32_t* sink = nullptr;
  if (cudaMalloc((void**)&buf, bytes) != cudaSuccess || cudaMalloc((void**)&sink, 148 * 8 * 4) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(buf);
    return fail(ctx, RB_ENOMEM, "cudaMalloc (read bandwidth scratch)");
  }
  cudaStream_t s = ctx->stream;
  cudaError_t e = cudaMemsetAsync(buf, 0, bytes, s);
  float best = 1e30f;
  for (int r = 0; r < repeats + 2 && e == cudaSuccess; ++r) {   // two untimed launches first
    if ((e = cudaEventRecord(ctx->ev[0], s)) != cudaSuccess) break;
    if ((e = launch_read_stream(buf, bytes, sink, s)) != cudaSuccess) break;
    if ((e = cudaEventRecord(ctx->ev[1], s)) != cudaSuccess) break;
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) break;
    float ms = 0.0f;
    if ((e = cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1])) != cudaSuccess) break;
    if (r >= 2 && ms < best) best = ms;
  }
  cudaFree(buf);
  cudaFree(sink);
  if (e != cudaSuccess) return fail(ctx, RB_ECUDA, "rb_testing_read_bandwidth", e);
  *gb_per_s = (double)bytes / (best * 1e-3) / 1e9;
  return RB_OK;
}

int64_t rb_launch_count(const rb_ctx* ctx) { return ctx ? ctx->launches : 0; }

rb_status rb_sync(rb_ctx* ctx) {
  if (!ctx) return RB_EINVAL;
  CK(cudaStreamSynchronize(ctx->stream));
  return RB_OK;
}

const char* rb_last_error(const rb_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

void rb_destroy(rb_ctx* ctx) {
  if (!ctx) return;
  if (ctx->sstage) cudaStreamSynchronize(ctx->sstage);
  if (ctx->front) cudaStreamSynchronize(ctx->front);
  if (ctx->front2) cudaStreamSynchronize(ctx->front2);
  if (ctx->stream) cudaStreamSynchronize(ctx->stream);
  drop_graphs(ctx);
  void* ptrs[] = {ctx->bank, ctx->bank_quality, ctx->bank_outlen, ctx->arena, ctx->q32, ctx->q32_in, ctx->qs, ctx->part_sim,
                  ctx->gthr, ctx->bank32, ctx->scratch_nn_idx, ctx->scratch_nn_sim, ctx->scores, ctx->scores0, ctx->f_nodes,
                  ctx->f_root, ctx->f_begin, ctx->f_nbegin, ctx->f_base, ctx->dev_clock, ctx->sweep_buf, ctx->f_cwords, ctx->f_cbegin};
  for (void* p : ptrs) cudaFree(p);
  for (int j = 1; j < kSlots; ++j) {
    cudaFree(ctx->slot[j].qs);
    cudaFree(ctx->slot[j].part_sim);
    cudaFree(ctx->slot[j].q32);
    cudaFree(ctx->slot[j].gthr);
  }
  for (auto& sl : ctx->slot) {
    if (sl.ev_stage) cudaEventDestroy(sl.ev_stage);
    if (sl.ev_front) cudaEventDestroy(sl.ev_front);
    if (sl.ev_back) cudaEventDestroy(sl.ev_back);
  }
  if (ctx->front) cudaStreamDestroy(ctx->front);
  if (ctx->front2) cudaStreamDestroy(ctx->front2);
  if (ctx->sstage) cudaStreamDestroy(ctx->sstage);
  if (ctx->ev_bigfin) cudaEventDestroy(ctx->ev_bigfin);
  for (auto& e : ctx->ev)
    if (e) cudaEventDestroy(e);
  if (ctx->h_zc) cudaFreeHost(ctx->h_zc);
  for (auto& A : ctx->async)
    if (A.h) cudaFreeHost(A.h);
  if (ctx->own_stream) cudaStreamDestroy(ctx->stream);
  delete ctx;
}

}  // extern "C"
