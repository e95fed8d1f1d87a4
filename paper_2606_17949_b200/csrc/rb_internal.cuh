// rb_internal.cuh -- declarations shared by the kernels and the C-ABI layer (product code).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace rb {

constexpr int kMaxK = 64;          // largest candidate list (k + rerank_slack)
constexpr int kMaxM = 16;          // model tiers
constexpr int kMaxI = 1024;        // instances
constexpr int kTileM = 128;        // queries per MMA tile (TMEM lanes)
constexpr int kTileN = 256;        // bank rows per MMA tile (TMEM columns of one accumulator)
constexpr int kBoxN = 64;          // bank rows per TMA box
constexpr int kSlots = 3;          // buffer sets of the throughput mode = decisions that can be in flight
constexpr int kSplitPlanes = 3;     // fp32 storage: bf16 columns per fp32 column in the scanned rows ([hi | mid | hi] x [hi | hi | mid])
constexpr int kRowUnit = 16;       // the single-CTA scan splits the bank over its CTAs in groups of this many rows
constexpr int kTileK = 64;         // bf16 per K chunk = one 128-byte swizzle row
constexpr int kMaxPendingAdvance = 4;   // rb_advance_state calls a decision can absorb (CallParams::adv_ms)

// Instance table + per-tier coefficients as the score/dispatch kernels see them (device memory).
struct InstTable {
  int32_t I, M;
  const int32_t* tier;     // [I]
  const int32_t* cap;      // [I]
  const float* price_in;   // [M]
  const float* price_out;  // [M]
  const float* pre;        // [M]
  const float* dec;        // [M]
  const float* slope;      // [M]
  const int32_t* present;  // [M] 1 if the tier has an instance
  const float* dec_i;      // [I] dec[tier[i]]   (per-instance copies: no dependent lookups in the dispatch loop)
  const float* slope_i;    // [I] slope[tier[i]]
};

// Gradient-boosted TPOT head (reading 9b) as the kernels see it (device memory).
constexpr int kMaxTreesPerTier = 256;
constexpr int kMaxFeatures = 8;
struct ForestDev {
  const int4* nodes;           // (feature, value bits, left, right); feature < 0: leaf.  Stored tier by tier:
  const int32_t* tier_node_begin;   // [M+1] tier t's nodes are nodes[tier_node_begin[t] .. tier_node_begin[t+1])
  int32_t max_tier_nodes;      // the largest tier's node count (shared-memory cache sizing)
  const int32_t* tree_root;    // [n_trees]
  const int32_t* tier_begin;   // [M+1]
  const float* base;           // [M]
  const float* aux;            // [I x (F-2)] auxiliary telemetry features
  const float* tpot0;          // [I] head evaluated on the batch-start state (tpot_kernel)
  int32_t n_features;
  // the forest again, packed for the dispatch loop's shared-memory cache: tier t's block = cwords[tier_cbegin[t] ..
  // tier_cbegin[t+1]) = [one root word per tree | nodes in pre-order]; an inner node is two words (threshold bits;
  // feature | left-is-leaf << 3 | right-is-leaf << 4 | (right child's offset - own offset) << 5), its left child follows
  // it; a leaf is one word (value bits); a root word = (offset in the block) << 1 | is-leaf
  const uint32_t* cwords;
  const int32_t* tier_cbegin;  // [M+1]
  int32_t total_cwords, max_tier_cwords;
  float tpot_hi;               // no evaluation of the head exceeds this (|base| + sum of the trees' largest |leaf|, doubled)
};

// Per-call parameters live in device memory so that a captured graph can be replayed with new weights and new
// caller buffers.  Every pointer is a DEVICE pointer: the caller's own buffer, or the context's staging buffer
// when the caller passed host memory.  Optional outputs are NULL when not wanted.
struct CallParams {
  float w_qual, w_lat, w_cost;
  int32_t commit;
  const float* query;      // [B x d] fp32 prompt embeddings
  const int32_t* plen;     // [B]
  const float* q_src;      // [B x M] predicted quality the score/dispatch stages consume
  const float* l_src;      // [B x M] predicted output length, likewise
  int32_t* assignment;     // [B]
  float* scores;           // [B x I] or NULL
  float* scores0;          // [B x I] or NULL
  int32_t* order;          // [B] or NULL
  float* pred_q;           // [B x M] or NULL: extra copy of the estimate for the caller
  float* pred_l;
  int32_t* nn_idx;         // [B x k] or NULL
  float* nn_sim;
  const float* budget;     // [B] per-request cost budgets (Eq. 2) or NULL: no admission filter
  int32_t* max_tokens;     // [B] or NULL: output-token clamp of the chosen instance
  uint32_t* done_flag;     // pinned host word or NULL: the dispatch kernel stores done_seq there once the assignment is out
  uint32_t done_seq;       //   (host callers wait on it instead of synchronising the stream)
  int32_t n_adv;           // pending rb_advance_state calls folded into this decision's dispatch kernel (<= kMaxPendingAdvance)
  float adv_ms[4];         // their elapsed_ms, in call order
  const float* sweep_w;    // weight sweep (rb_sweep_weights): [P x 3] weights, point p = the CTA's grid coordinate; the
                           //   term, key and assignment arrays are then [P][...]; NULL: the w_* fields above
};

// Dispatch modes (rb_options; SURVEY 8(f) #2, P:L227 isolation arms, P:L266 ablations).
struct DispatchModes {
  int32_t lpt_enabled;     // 1: LPT order; 0: input order
  int32_t update_mode;     // 0: none; 1: d += L^ and b = min(b+1, cap) (default); 2: d only (P:L121 literally)
  int32_t tiebreak_mode;   // 0: (S desc, d asc, i asc) reactive shortest queue; 1: (S desc, T^ asc, i asc) predictive
  int32_t latency_mode;    // 0: live linear head over the dead-reckoned state; 1: static prior T^ = dec * L^ (arm 4);
                           // 2: live gradient-boosted head (ForestDev)
};

#ifdef __CUDACC__
// Leaf of one tree for the features (x0 = running, x1 = queued tokens, x2.. = aux): XGBoost's rule, left iff x < threshold.
__device__ __forceinline__ float forest_leaf(const int4* __restrict__ nodes, int root, float xb, float xd,
                                             const float* __restrict__ aux_i) {
  int4 nd = __ldg(&nodes[root]);
  while (nd.x >= 0) {
    const float x = nd.x == 0 ? xb : (nd.x == 1 ? xd : __ldg(&aux_i[nd.x - 2]));
    nd = __ldg(&nodes[(x < __int_as_float(nd.y)) ? nd.z : nd.w]);
  }
  return __int_as_float(nd.y);
}
// Leaves of trees tr0 + lane, tr0 + lane + 32, ... < tr1 into out[tree - tr0]: every lane walks up to four trees at once
// (a walk is a chain of dependent node loads; four independent chains hide most of their latency).
__device__ __forceinline__ void forest_leaves_warp(const int4* __restrict__ nodes, const int32_t* __restrict__ tree_root,
                                                   int tr0, int tr1, int lane, float xb, float xd,
                                                   const float* __restrict__ aux_i, float* out) {
  for (int base = tr0 + lane; base < tr1; base += 128) {
    int4 nd[4];
    bool live[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      live[u] = base + 32 * u < tr1;
      nd[u] = live[u] ? __ldg(&nodes[__ldg(&tree_root[base + 32 * u])]) : make_int4(-1, 0, 0, 0);
    }
    while ((nd[0].x >= 0) | (nd[1].x >= 0) | (nd[2].x >= 0) | (nd[3].x >= 0)) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (nd[u].x >= 0) {
          const float x = nd[u].x == 0 ? xb : (nd[u].x == 1 ? xd : __ldg(&aux_i[nd[u].x - 2]));
          nd[u] = __ldg(&nodes[(x < __int_as_float(nd[u].y)) ? nd[u].z : nd[u].w]);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (live[u]) out[base + 32 * u - tr0] = __int_as_float(nd[u].y);
  }
}
#endif

// ---- programmatic dependent launch ---------------------------------------------------------------------------
// Consecutive kernels of one decision are chained with programmatic stream serialization: a kernel lets its
// successor start (launch_dependents, first thing) so that the successor's launch latency and prologue overlap
// with it, and waits (grid_dependency_wait) before it touches anything its predecessor produces.  Both are
// no-ops for a kernel launched without the attribute.
#ifdef __CUDACC__
// ---- mbarrier / bulk-copy PTX wrappers shared by the scan kernels and the finishing code --------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred P1;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, P1;\n\t}"
        : "=r"(ok)
        : "r"(addr), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
// 1-D bulk copy global -> shared (bytes a multiple of 16, both addresses 16-byte aligned), completion on an mbarrier.
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// a4: per-(request, tier) term A[m] = w_q*Q^ + w_c*(1 - C/Cmax) of Eq. 1, with the admission filter of
// Eq. 2: tier m is a candidate iff it has an instance and C[m] <= budget; if no tier fits, the cheapest
// present tiers are the candidates (reading 24).  Cmax runs over the candidates ("normalized by their
// candidate maxima").  Non-candidates get A = -inf, which the score and dispatch kernels read as "filtered out".
// Also returns the LPT key max_m L^ over present tiers (budgets do not enter it).
// Warp-collective: all 32 lanes call it; lane j < M carries tier j's cost C and predicted length L (other lanes are
// ignored: their bit of `present` is clear), present: bit j set iff tier j has an instance.  The maxima and the minimum
// over tiers are warp reductions on the order-preserving integer image of the floats (max and min are exact, so the
// result equals a sequential scan over the tiers); returns lane j's A[j].
__device__ __forceinline__ uint32_t rb_f2o(float f) {   // larger float <=> larger uint
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float rb_o2f(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
__device__ __forceinline__ float tier_term_A_warp(int lane, uint32_t present, float C, float L, float Q, float wq, float wc,
                                                  bool has_budget, float budget, float* key_out) {
  const bool here = (present >> lane) & 1u;
  const uint32_t okmax = __reduce_max_sync(0xffffffffu, here ? rb_f2o(L) : 0u);
  const uint32_t ocmin = __reduce_min_sync(0xffffffffu, here ? rb_f2o(C) : 0xffffffffu);
  const float kmax = present ? rb_o2f(okmax) : 0.0f, Cmin = present ? rb_o2f(ocmin) : 0.0f;
  const bool fits = here && (!has_budget || C <= budget);
  const bool any = __any_sync(0xffffffffu, fits);
  const bool cand = any ? fits : (here && C == Cmin);
  const uint32_t ocmax = __reduce_max_sync(0xffffffffu, cand ? rb_f2o(C) : 0u);
  const float Cmax = __any_sync(0xffffffffu, cand) ? rb_o2f(ocmax) : 0.0f;
  *key_out = __fadd_rn(kmax, 0.0f);   // -0 -> +0 so that the sort key order equals float order
  if (!cand) return -INFINITY;
  const float ct = (Cmax > 0.0f) ? __fsub_rn(1.0f, __fdiv_rn(C, Cmax)) : 0.0f;
  return __fadd_rn(__fmul_rn(wq, Q), __fmul_rn(wc, ct));
}

template <typename... KArgs, typename... Args>
cudaError_t launch_chained(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// ---- launchers (each returns the cudaError of its launch) ---------------------------------------------
// plain streaming read of `bytes` bytes (rb_testing_read_bandwidth); sink: 148 * 8 words
cudaError_t launch_read_stream(const void* buf, size_t bytes, uint32_t* sink, cudaStream_t s);
// fp32 -> bf16 (RNE), n elements (bank conversion in rb_create).
cudaError_t launch_convert_bf16(const float* in, __nv_bfloat16* out, size_t n, cudaStream_t s);

// a0: cp->query (fp32) -> bf16 staging [Bpad x d]; rep copies of the B queries at rows j*(128/rep) + r (rep > 1 only
// when Bpad = 128), all other rows zero.  Also clears gthr [n_gthr] (the scan's cross-slab thresholds).
// split = 1 (fp32 storage): rows of kSplitPlanes d columns [hi | hi | mid] of the two-plane bf16 split of every value.
cudaError_t launch_stage_queries(const CallParams& cp, __nv_bfloat16* qs, int B, int Bpad, int d, int rep, uint32_t* gthr,
                                 int n_gthr, int split, float* q32 /* split: device copy of the B fp32 rows */, cudaStream_t s);
// fp32 bank rows -> [hi | mid | hi] bf16 rows of kSplitPlanes d columns (fp32 storage: the bank the tensor-core scan reads)
cudaError_t launch_split_bank(const float* in, __nv_bfloat16* out, size_t rows, int d, cudaStream_t s);
// query replicas over the TMEM lane quarters: 4 (B <= 32), 2 (B <= 64), 1; halved while the finishing kernel could not
// hold max_grid * replicas lists of kcap entries in shared memory (long lists: k = 32)
int scan_tc_replicas(int B, int kcap, int max_grid);

// a1 (bf16): tcgen05 scan.  The lists (sim fp32 / idx int32, idx -1 = empty, each sorted by (sim desc, idx asc)) are
// written through part_sim as QUERY-MAJOR 32-byte records: record ((r * nlists + list) * KCAP/4 + quad) =
// [4 similarities | 4 indices], nlists = grid * rep; part_sim must have room for nlists * Bpad * KCAP * 8 bytes.  Returns the grid size used through *grid_out.  kcap in {4,8,16,32,64}; bank
// rows are split over the CTAs in units of kRowUnit rows: CTA c owns units [units*c/grid, units*(c+1)/grid);
// tm_bank16: the bank again with 16-row boxes (the remainder of a CTA's last tile).
cudaError_t launch_scan_tc(const CUtensorMap* tm_q, const CUtensorMap* tm_bank, const CUtensorMap* tm_bank16, int64_t N, int d, int B, int Bpad,
                           int kcap, int max_grid, float* part_sim, int32_t* part_idx, int* grid_out,
                           unsigned long long* dev_clock /* NULL, or [2] = {~0, 0}: earliest CTA start / latest CTA end (globaltimer ns) */,
                           cudaStream_t s);
size_t scan_tc_smem_bytes();
cudaError_t scan_tc_prepare();  // opt in to the dynamic shared memory size; call once

// a1 (bf16, B > 128): the same scan on CTA pairs (tcgen05 cta_group::2, 256 queries x 256 bank rows per MMA tile).
// Bpad is a multiple of 256.  part_* are [clusters][Bpad][KCAP]; cluster c owns the 256-row tiles
// [tiles*c/clusters, tiles*(c+1)/clusters).  Returns the number of clusters through *clusters_out.
// gthr [(1 + clusters) x Bpad] must be zero at launch (launch_stage_queries clears it): cross-slab admission
// thresholds ([Bpad] best K-th best of any slab, then per slab the (kc+15)/16-th best it has seen so far).
cudaError_t launch_scan_tc2(const CUtensorMap* tm_q, const CUtensorMap* tm_bank, int64_t N, int d, int B, int Bpad,
                            int kcap, int kc, int max_grid, float* part_sim, int32_t* part_idx, uint32_t* gthr,
                            int* clusters_out, cudaStream_t s);
int scan_tc2_clusters(int64_t N, int max_grid);
cudaError_t scan_tc2_prepare();

// a2 + a3 (+ a4 when with_terms): one CTA per query merges the nlists sorted partial lists
// (part_* [nlists][Bpad][kcap]) into the kc best, re-ranks them exactly (bf16 storage, rerank != 0), keeps k,
// aggregates the labels with distance weights and, when with_terms, derives the per-(request, tier) terms
// A, P and the LPT key.  pred_q / pred_l are the context's [B x M] buffers; copies for the caller go through cp.
struct FinishArgs {
  const float* part_sim;
  const int32_t* part_idx;
  int nlists, kcap, Bpad, kc, k;   // nlists = grid * lists_per_cta
  int lists_per_cta;
  int records;              // 1: part_sim holds the query-major 32-byte records of launch_scan_tc; 0: part_sim / part_idx
                            //    are [nlists][Bpad][kcap] arrays
  int slab_unit;            // rows per slab unit: slab c = rows [units*c/nslabs, units*(c+1)/nslabs) * slab_unit
  int64_t N;
  const __nv_bfloat16* bank;
  const __nv_bfloat16* qs;
  const float* bank32;      // fp32 storage: the fp32 bank rows the exact re-rank reads (rerank = 2) ...
  const float* q32;         // ... and the fp32 query rows (device copy made by the staging kernel)
  int d, rerank;            // rerank: 0 none, 1 exact from the bf16 rows (bf16 storage), 2 exact from the fp32 rows
  int rescan;               // 1: lists are shorter than kc -> slabs whose list was popped completely are searched again
  const float* bank_quality;
  const float* bank_outlen;
  int M, weight_mode;
  float eps;
  int with_terms;
  float* pred_q;
  float* pred_l;
  float* termA;
  float* termP;
  float* key;
};
cudaError_t launch_finish(const FinishArgs& a, InstTable t, const CallParams& cp, int B, cudaStream_t s);
int estimate_cp_arg(const void* func, int* nargs);   // which argument of a kernel of estimate.cu holds the CallParams (-1: none)
int dispatch_cp_arg(const void* func, int* nargs);   // likewise for score_dispatch.cu
size_t finish_smem_bytes(int nlists, int kcap, int kc, int d, int rerank);
cudaError_t finish_prepare(size_t max_smem);

// a4+a5 from caller-supplied predictions (cp->q_src, cp->l_src): per-(request, tier) terms, LPT keys and the
// batch-start score matrix (cp->scores0 when non-NULL).
cudaError_t launch_score(InstTable t, const float* dq, const int32_t* bq, const CallParams& cp, int B, float* termA,
                         float* termP, float* key, DispatchModes modes, ForestDev forest, cudaStream_t s, int points = 1);

// a6+a7: LPT sort + greedy dispatch with dead-reckoned updates, one CTA.
cudaError_t launch_lpt_dispatch(InstTable t, float* dq, int32_t* bq, const float* termA, const float* termP,
                                const float* key, const CallParams& cp, int B, DispatchModes modes, ForestDev forest,
                                cudaStream_t s, int points = 1);

cudaError_t lpt_dispatch_prepare();  // opt in to the dynamic shared memory size; call once

// a4..a7 from caller-supplied predictions (cp->q_src, cp->l_src) with the terms and keys in a file-scope __device__ array
// of score_dispatch.cu instead of allocated buffers (rb_decide_from_predictions_static): B <= static_scratch_max_b() and
// B * M <= static_scratch_max_bm(), else cudaErrorInvalidValue.  Allocates nothing.
int static_scratch_max_b();
int static_scratch_max_bm();
cudaError_t launch_score_dispatch_static(InstTable t, float* dq, int32_t* bq, const CallParams& cp, int B, DispatchModes modes,
                                         ForestDev forest, cudaStream_t s);

// Boosted head over the current state: tpot_out[i] = max(base + sum of leaves (fp32, tree order), 1e-6) for every
// instance (one CTA per instance, one thread per tree, sequential sum by thread 0).  elapsed_ms >= 0: also applies
// the a8 drain rule with that tpot (rb_advance_state under latency_mode 2).
cudaError_t launch_tpot_forest(InstTable t, ForestDev forest, float* dq, int32_t* bq, float* tpot_out, float elapsed_ms,
                               cudaStream_t s);

// Counts pairs on which the dispatch loop's branch-free division differs from the IEEE one (must be 0).
cudaError_t launch_div_selftest(unsigned long long n, unsigned long long seed, unsigned long long* mismatches, cudaStream_t s);

// Batch-level matching replay: quota-constrained optimum of sum_r S0[r, a(r)], one CTA.
// All pointers device; *status = 1 when no feasible assignment exists.
cudaError_t launch_match_replay(const float* S0, int B, int I, const int32_t* quota, const int32_t* greedy, int32_t* match,
                                double* objective, int32_t* n_diverged, int32_t* status, cudaStream_t s);
cudaError_t match_replay_prepare();

// Pipeline-mode dispatchers, one warp; members / tstart: instances sorted by (tier, index) and the start of each
// tier's run; counter / cursor: device-resident draw counter and per-tier round-robin cursors.
cudaError_t launch_pipeline_dispatch(InstTable t, const int32_t* members, const int32_t* tstart, float* dq, int32_t* bq,
                                     const int32_t* model, const float* outlen, int B, int policy, unsigned long long seed,
                                     unsigned long long* counter, int32_t* cursor, int commit, int32_t* assignment,
                                     cudaStream_t s);

// Adaptive batch size (reading 27): *target = bs_min + floor((bs_max - bs_min) * n_busy / I), n_busy = #{b_i >= cap_i}.
cudaError_t launch_batch_target(InstTable t, const int32_t* bq, int bs_min, int bs_max, int32_t* target, int32_t* n_busy,
                                cudaStream_t s);

// a8: dead reckoning between batches.
cudaError_t launch_advance(InstTable t, float* dq, int32_t* bq, float elapsed_ms, cudaStream_t s);

}  // namespace rb
