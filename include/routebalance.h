/*
 * routebalance.h -- C ABI of the B200-native RouteBalance per-batch scheduling decision.
 *
 * What the library computes (citations: P:Lnnn = line nnn of the paper text PAPER.md,
 * "RouteBalance: Fused Model Routing and Load Balancing for Heterogeneous LLM Serving"):
 *
 *   estimate  (§4.2 "Model estimator"):  k-nearest labelled prompts of every query embedding in a
 *             reference bank; distance-weighted per-model predicted quality Q^[r,m] and expected output
 *             length L^[r,m].
 *   latency   (§4.2 "Latency heads"):    T^[r,i] = T^tpot_i * (d_i/b_i + L^[r,m(i)]); the wait term
 *             d_i/b_i is dropped when instance i has a free decode slot.
 *   cost      (Eq. 2):                 C^[r,i] = l_r * c_in[m(i)] + L^[r,m(i)] * c_out[m(i)].
 *   score     (Eq. 1):                 S[r,i] = w_qual*Q^ + w_cost*(1 - C^/max_j C^) + w_lat*(1 - T^/max_j T^).
 *   dispatch  (§4.1, "Dead reckoning"): requests in LPT order (key max_m L^[r,m], longest
 *             first); each takes argmax_i S[r,i]; the chosen instance's local decode state grows by L^
 *             before the next request is scored.
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  The exact operation
 * order (one IEEE binary32 round-to-nearest operation per line, never fused) is stated in DESIGN.md
 * "Canonical arithmetic"; readings of the paper where it is silent are listed in DESIGN.md "Readings".
 *
 * Conventions for every call
 *   - Pointers marked [host|device] may be either; they are classified with cudaPointerGetAttributes.
 *     Pointers marked [host] must be host memory.
 *   - Input buffers are consumed before the call returns (host pointers) or in stream order on the
 *     context's stream (device pointers).  The library never keeps a caller pointer.
 *   - Outputs to host pointers are complete when the call returns; outputs to device pointers are complete
 *     in stream order on the context's stream.  (rb_decide with host buffers returns as soon as the assignment has
 *     reached host memory; work it queued behind that -- nothing a caller can observe -- may still be draining.)
 *   - All matrices are dense row-major.  Optional outputs may be NULL.
 *   - On any non-RB_OK return nothing the caller can observe has changed, except rb_last_error().
 *   - One context = one CUDA stream = one caller thread at a time.  Several contexts may coexist.
 */
#ifndef ROUTEBALANCE_H_
#define ROUTEBALANCE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rb_ctx rb_ctx; /* opaque; owns all device memory it uses */

typedef enum {
  RB_OK = 0,
  RB_EINVAL = 1,       /* bad argument (size, range, NULL, non-finite coefficient) */
  RB_ECUDA = 2,        /* a CUDA runtime/driver call failed; see rb_last_error */
  RB_ENOMEM = 3,       /* host or device allocation failed */
  RB_ESTATE = 4,       /* call order violated (e.g. rb_decide before rb_set_instances) */
  RB_EUNSUPPORTED = 5  /* valid request this build cannot serve (e.g. no sm_100 device) */
} rb_status;

typedef enum { RB_F32 = 0, RB_BF16 = 1 } rb_dtype;

/* Per-tier latency head.  The paper's head is a gradient-boosted TPOT regressor per (model, GPU) tier
 * (P:L119); its trained trees are not available, so the head is the linear stand-in of BASELINE.json:
 *   tpot_i = decode_ms_per_tok * (1 + batch_slope * b_i)      [ms per output token]
 *   T^[r,i] = prefill_ms_per_tok * l_r + tpot_i * (wait_i + L^[r,tier(i)])
 * prefill_ms_per_tok = 0 recovers the paper's formula exactly. */
typedef struct {
  float prefill_ms_per_tok;
  float decode_ms_per_tok;
  float batch_slope;
} rb_lat_head;

typedef struct {
  int32_t bank_dtype;     /* rb_dtype of bank_emb as passed to rb_create.                 default RB_F32  */
  int32_t store_dtype;    /* rb_dtype the bank is stored and searched in.                 default RB_BF16 */
                          /* RB_BF16: bank and queries are rounded to bf16 (RNE) once; similarity is the   */
                          /* dot product of the rounded values (tcgen05 tensor-core scan).                 */
                          /* RB_F32: the similarity is the dot product of the fp32 values.  The bank is also kept  */
                          /* as a two-plane bf16 split (x ~ hi + mid, three column blocks) that the same tensor-core  */
                          /* scan reads (candidates good to ~1e-5); the k + slack candidates are then re-ranked       */
                          /* exactly from the fp32 rows.  10 bytes per value: meant for small banks.                  */
  int32_t weight_mode;    /* 0: inverse distance 1/(dist+eps) ("distance-weighted"); 1: uniform     */
  float dist_eps;         /* eps above.                                                   default 1e-6    */
  int32_t rerank_slack;   /* the scan keeps k+slack candidates per query, their similarities are recomputed       */
                          /* exactly (fp64 accumulate) and the best k kept.                default 6       */
                          /* RB_F32 always re-ranks: 0 is read as min(6, 64 - k).                          */
                          /* 0: no re-rank; similarities are the tensor core's fp32 sums (within 4e-6), and  */
                          /* inverse-distance weights amplify that as a neighbour's similarity nears 1.      */
  int32_t lpt_enabled;    /* 1: dispatch in LPT order; 0: in input order.         default 1       */
  int32_t update_enabled; /* dead-reckoning update after each dispatch: 1: d += L^ and the decode batch   */
                          /* grows by one while a slot is free (default); 2: d only (P:L121 literally); 0: none   */
  int32_t max_batch;      /* largest B any later call may pass (scratch sizing).          default 4096    */
  int32_t use_graph;      /* 1: replay the decision as a captured CUDA graph.             default 1       */
  int32_t scan_list;      /* RB_BF16 only: entries the bank scan keeps per (CTA, query): 4|8|16|32|64, or 0 = */
                          /* chosen from the bank size.  Lists shorter than k+slack are exact all the same:  */
                          /* a slab whose list might hide neighbours is searched again.   default 0       */
  int32_t tiebreak_mode;  /* ties of the argmax over S: 0 (default): smaller queued_tokens d_i, then smaller i --  */
                          /* "the scheduler's reactive shortest-queue tiebreak" (P:L227 arm 2); 1: smaller T^[r,i], */
                          /* then smaller i -- "a predictive T^-argmin tiebreak" (arm 3)                           */
  int32_t latency_mode;   /* 0 (default): live linear latency head over the dead-reckoned state;         */
                          /* 2: live gradient-boosted TPOT head (rb_set_tpot_forest) in place of the linear one;   */
                          /* 1: static per-tier prior T^ = decode_ms_per_tok * L^ ("nominal TPOT x predicted       */
                          /* length; zero telemetry", P:L227 arm 4): no wait, batch-slope or prefill term          */
  int32_t pipeline;       /* 1: consecutive rb_decide calls with DEVICE buffers overlap -- the bank scan of a call runs on  */
                          /* an internal stream (its query staging on another, beside the scan before it) while the      */
                          /* finishing and dispatch stages of the call before it run on the context's stream (above 128  */
                          /* requests: the dispatch stage only).  Device inputs of                                       */
                          /* rb_decide must then be COMPLETE when the call is made (they are not ordered after earlier   */
                          /* work on the context's stream); outputs stay in stream order.  Results are those of the      */
                          /* unpipelined calls, bit for bit.  Three sets of per-decision buffers are kept.  default 0    */
  void* stream;           /* cudaStream_t all work is ordered on; NULL = legacy default stream            */
} rb_options;

/* Fills *opt with the defaults listed above.  opt [host]. */
void rb_options_default(rb_options* opt);

/* Creates a context holding the reference bank (N labelled prompts, d-dim embeddings, per-model
 * quality label in [0,1] and output length for each of M models).
 *   bank_emb      [host|device] N x d, dtype opt->bank_dtype (fp32, or bf16 as raw uint16)
 *   bank_quality  [host|device] N x M fp32
 *   bank_outlen   [host|device] N x M fp32
 *   k             neighbours per query, 1 <= k <= 64, k + rerank_slack <= 64, k <= N
 *   d             must be a multiple of 8; M in [1,16]; N < 2^31
 * The bank is copied (and converted to store_dtype); the caller may free its buffers on return.
 * Errors: RB_EINVAL on bad sizes/NULL, RB_EUNSUPPORTED without an sm_100 device, RB_ENOMEM, RB_ECUDA. */
rb_status rb_create(rb_ctx** out, const void* bank_emb, const float* bank_quality,
                    const float* bank_outlen, int64_t N, int32_t d, int32_t M, int32_t k,
                    const rb_options* opt /* NULL = defaults */);

/* Defines the instance set I (fixed at runtime; Table 1) and resets the dead-reckoned
 * state to (queued_tokens = 0, running = 0).
 *   tier      [host] I entries in [0,M): model/tier served by instance i, m(i)
 *   cap       [host] I entries >= 1: decode slots of instance i ("free decode slot" <=> running < cap)
 *   price_in  [host] M entries >= 0: price per input token of tier m (any unit; only ratios matter)
 *   price_out [host] M entries >= 0
 *   heads     [host] M latency heads, coefficients finite and >= 0
 *   1 <= I <= 1024.  May be called again at any time between decisions (tier loss). */
rb_status rb_set_instances(rb_ctx* ctx, int32_t I, const int32_t* tier, const int32_t* cap,
                           const float* price_in, const float* price_out, const rb_lat_head* heads);

/* Gradient-boosted TPOT head ("For each (model, GPU) tier we train one XGBoost TPOT head ... one XGBoost call
 * per tier (not per instance)").  The trained boosters of the paper are not available: the forest is an input, and
 * what the library implements is the evaluation rule of an XGBoost regression forest (reading 9b):
 *   features of instance i  x[0] = (float)running_i, x[1] = queued_tokens_i (both dead-reckoned within a batch),
 *                           x[2+j] = aux[i,j]: further telemetry (queue depth, KV-cache pressure, recent
 *                           service rate), constant during a batch, set with rb_set_telemetry (default 0)
 *   node                    feature >= 0: go to `left` if x[feature] < value, else to `right`; feature < 0: leaf `value`
 *   tier t                  p = base[t]; for each tree of the tier in order: p = p + leaf   (fp32);  tpot = max(p, 1e-6)
 * Used when rb_options.latency_mode = 2: tpot_i replaces decode_ms_per_tok*(1+batch_slope*b_i) in T^ and in
 * rb_advance_state; the chosen instance's head is evaluated again after every dispatch.
 *   nodes            [host] n_nodes; children of an internal node must have larger indices than the node
 *   tree_root        [host] n_trees node indices
 *   tier_tree_begin  [host] M+1: trees of tier t are tree_root[tier_tree_begin[t] .. tier_tree_begin[t+1]), <= 256 each
 *   base             [host] M;  n_features = 2 + (aux columns), in [2,8]
 * Errors: RB_EINVAL (ranges, non-finite values, backward links), RB_ENOMEM.  Decisions under latency_mode 2 return
 * RB_ESTATE until a forest is set. */
typedef struct {
  int32_t feature;
  float value;
  int32_t left;
  int32_t right;
} rb_tree_node;
rb_status rb_set_tpot_forest(rb_ctx* ctx, const rb_tree_node* nodes, int32_t n_nodes, const int32_t* tree_root,
                             int32_t n_trees, const int32_t* tier_tree_begin, const float* base, int32_t n_features);

/* Auxiliary telemetry features of the boosted head: aux [host|device] I x (n_features - 2) fp32, row i = instance i.
 * Reset to 0 by rb_set_instances.  RB_ESTATE before rb_set_instances / rb_set_tpot_forest. */
rb_status rb_set_telemetry(rb_ctx* ctx, const float* aux);

/* Seeds the dead-reckoned state from telemetry: queued_tokens[i] = pending decode tokens
 * d_i >= 0 (finite), running[i] = decode batch size b_i >= 0.  Both [host|device], I entries. */
rb_status rb_set_state(rb_ctx* ctx, const float* queued_tokens, const int32_t* running);

/* Reads the current dead-reckoned state back.  Both [host|device], I entries; either may be NULL. */
rb_status rb_get_state(rb_ctx* ctx, float* queued_tokens, int32_t* running);

/* Dead reckoning between batches (BASELINE.json; the drain rule is this library's, reading 22):
 * every instance with b_i > 0 drains d_i <- max(0, d_i - b_i * elapsed_ms / tpot_i); b_i <- 0 when d_i
 * reaches 0.  elapsed_ms must be finite and >= 0.
 * The drain is applied in stream order before anything reads or writes the state; under the linear head it is deferred
 * into the first kernel of the next rb_decide (no launch of its own), other calls apply it first. */
rb_status rb_advance_state(rb_ctx* ctx, float elapsed_ms);

/* Adaptive batch size (§4.1: "Batch size is adaptive -- larger when more instances are busy, smaller when idle";
 * P:L191 §6.3: "Adaptive sizing ties t_form to cluster busyness").  The paper states no rule; this library's
 * (reading 27), evaluated on the current dead-reckoned state (pending rb_advance_state calls applied first):
 *   an instance is busy when it has no free decode slot, running_i >= cap_i (the condition of the wait term);
 *   n_busy = number of busy instances;   target = bs_min + floor((bs_max - bs_min) * n_busy / I).
 * An idle cluster gives bs_min, a saturated one bs_max; bs_min = bs_max is the fixed batch size of the paper's
 * "adaptive-off" ablation.  A stream driver closes the next batch when it holds `target` requests (or its first
 * request has waited long enough) -- paper_2606_17949_b200/stream.py is one.
 *   target  [host|device] 1 int32;   n_busy [host|device] 1 int32 or NULL
 * 1 <= bs_min <= bs_max, else RB_EINVAL.  Host outputs synchronise the context's stream. */
rb_status rb_batch_target(rb_ctx* ctx, int32_t bs_min, int32_t bs_max, int32_t* target, int32_t* n_busy);

/* One per-batch decision: estimate -> score -> LPT greedy dispatch, committing the dead-reckoned updates.
 *   query_emb    [host|device] B x d fp32 prompt embeddings (unit norm expected, not enforced)
 *   prompt_len   [host|device] B int32 input token counts l_r >= 0
 *   w            [host] (w_qual, w_lat, w_cost), each >= 0, |sum - 1| <= 1e-5
 *   assignment   [host|device] B int32: chosen instance per request (indexed like the input batch); -1 = no admissible
 *                instance, which only non-finite inputs can produce (a NaN label, prediction, price or budget makes every
 *                cost comparison of the request false); labels, predictions and budgets are not checked for finiteness
 *   scores       [host|device] B x I fp32 or NULL: row r = S[r,:] as seen when r was dispatched
 *   pred_quality [host|device] B x M or NULL; pred_outlen likewise
 *   nn_idx       [host|device] B x k int32 or NULL: neighbours, best first (similarity desc, index asc)
 *   nn_sim       [host|device] B x k fp32 or NULL
 * 1 <= B <= max_batch.  RB_ESTATE before rb_set_instances. */
rb_status rb_decide(rb_ctx* ctx, const float* query_emb, const int32_t* prompt_len, int32_t B,
                    const float w[3], int32_t* assignment, float* scores, float* pred_quality,
                    float* pred_outlen, int32_t* nn_idx, float* nn_sim);

/* rb_decide for a serving loop that keeps up to three decisions in flight (needs rb_options.pipeline = 1): rb_decide_submit copies
 * the batch into pinned memory the kernels read in place, enqueues the decision and returns at once; rb_decide_collect
 * waits for the OLDEST submitted decision and copies its assignment out (the dispatch kernel writes it, then a completion
 * word, into pinned host memory).  The usual loop is submit(j + 2); collect(j): the host side of one decision and the bank
 * scan of the next overlap the finishing and dispatch stages of the one before (with only submit(j + 1); collect(j) the
 * rate is half a decision's latency, not the scan's duration).  rb_advance_state calls made before a
 * submission are applied by that decision, in order, exactly as with rb_decide; results equal rb_decide's bit for bit.
 *   query_emb   [host] B x d fp32;   prompt_len [host] B int32;   1 <= B <= min(128, max_batch)
 *   assignment  [host] B int32 (rb_decide_collect; B must be the submitted batch's)
 * RB_ESTATE: a fourth submission with three in flight, a collect with none, pipeline = 0.  RB_EUNSUPPORTED: boosted latency
 * head, graph replay off, no mapped pinned memory. */
rb_status rb_decide_submit(rb_ctx* ctx, const float* query_emb, const int32_t* prompt_len, int32_t B, const float w[3]);
rb_status rb_decide_collect(rb_ctx* ctx, int32_t* assignment, int32_t B);

/* rb_decide with the per-request cost budgets of Eq. 2: "a pre-scoring filter keeps only candidates whose
 * predicted total cost (input tokens plus KNN-predicted output length, at the model's rates) fits within it":
 * the candidates of request r are the instances i with C^[r,i] = l_r*c_in[m(i)] + L^[r,m(i)]*c_out[m(i)] <= budget[r];
 * the maxima of Eq. 1 and the argmax run over the candidates; if nothing fits, the cheapest instances are the
 * candidates (the paper is silent; reading 24).  Filtered instances are reported with S = -inf.
 *   budget      [host|device] B fp32, same unit as price * tokens; +inf = unconstrained; NULL = no filter (rb_decide)
 *   max_tokens  [host|device] B int32 or NULL: floor((budget[r] - l_r*c_in)/c_out) at the chosen model's prices,
 *               clamped to [0, 2147483520] -- the dispatch-time clamp of P:L97 ("max_tokens clamped to the remaining
 *               budget"); INT32_MAX where budget[r] is +inf (or c_out = 0 and the prompt fits)
 * Budgets must not be NaN.  Everything else as rb_decide. */
rb_status rb_decide_budgeted(rb_ctx* ctx, const float* query_emb, const int32_t* prompt_len, const float* budget,
                             int32_t B, const float w[3], int32_t* assignment, int32_t* max_tokens, float* scores,
                             float* pred_quality, float* pred_outlen, int32_t* nn_idx, float* nn_sim);

/* The score + dispatch stages alone, from caller-supplied predictions (quality, outlen: B x M fp32,
 * [host|device]).  commit = 0 leaves the dead-reckoned state untouched (weight sweeps from one state).
 *   scores0 [host|device] B x I or NULL: S[r,:] of every request evaluated from the batch-start state
 *   order   [host|device] B int32 or NULL: dispatch order (order[j] = request dispatched j-th) */
rb_status rb_decide_from_predictions(rb_ctx* ctx, const float* quality, const float* outlen,
                                     const int32_t* prompt_len, int32_t B, const float w[3],
                                     int32_t commit, int32_t* assignment, float* scores,
                                     float* scores0, int32_t* order);

/* rb_decide_from_predictions with budgets; budget / max_tokens as in rb_decide_budgeted. */
rb_status rb_decide_from_predictions_budgeted(rb_ctx* ctx, const float* quality, const float* outlen,
                                              const int32_t* prompt_len, const float* budget, int32_t B, const float w[3],
                                              int32_t commit, int32_t* assignment, int32_t* max_tokens, float* scores,
                                              float* scores0, int32_t* order);

/* rb_decide_from_predictions for callers that may not allocate (code inside a CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same score + dispatch stages (Eq. 1), launched
 * directly on the context's stream, with the kernels' scratch -- the per-(request, tier) terms and the LPT keys -- in a
 * fixed __device__ array of the library (69,632 bytes per GPU that loads the library, held until the process exits)
 * instead of allocated buffers.  The call allocates nothing: no cudaMalloc / cudaFree, no graph capture or instantiation,
 * no staging copies, no stream synchronisation.
 *   quality, outlen  [device] B x M fp32;   prompt_len [device] B int32;   assignment [device] B int32 (-1 as rb_decide)
 *   w, commit        as rb_decide_from_predictions; pending rb_advance_state calls are applied first, as there
 * Limit: 1 <= B <= 1024 and B * M <= 8192; beyond it RB_EINVAL (rb_last_error names the limit), nothing launched.
 * RB_EINVAL also for a host pointer.  The array is ONE per GPU, shared by every context and every call, and keeps the last
 * call's contents (nothing in it has to start at zero: every word a call reads it has written first): calls that overlap
 * on the GPU -- two contexts on different streams, or threads -- race on it; calls on one stream do not.
 * Results equal rb_decide_from_predictions' bit for bit. */
rb_status rb_decide_from_predictions_static(rb_ctx* ctx, const float* quality, const float* outlen,
                                            const int32_t* prompt_len, int32_t B, const float w[3],
                                            int32_t commit, int32_t* assignment);

/* Weight sweep ("RouteBalance sweeps 16 weight tuples on the simplex"; "turning only the weight vector,
 * RouteBalance traces a monotone frontier"): P independent score + dispatch passes over the same predictions from the
 * same dead-reckoned state, one per weight vector, none committed.  Point p's result equals that of
 * rb_decide_from_predictions_budgeted(..., w + 3p, commit = 0, ...); the passes are independent, so they run
 * concurrently -- one CTA per point -- and a whole sweep costs about one pass.
 *   quality, outlen, prompt_len, budget   as rb_decide_from_predictions_budgeted (budget NULL: no filter)
 *   w           [host] P x 3 fp32 (qual, lat, cost per row), each row on the 3-simplex; 1 <= P <= 65535
 *   assignment  [host|device] P x B int32, row p = the assignment under w[p]
 * The state, the pipeline cursors and the captured graphs are left untouched.  Scratch of P*B*(2M+2)*4 bytes is kept
 * by the context (grown on demand, released by rb_destroy). */
rb_status rb_sweep_weights(rb_ctx* ctx, const float* quality, const float* outlen, const int32_t* prompt_len,
                           const float* budget, int32_t B, const float* w, int32_t P, int32_t* assignment);

/* Pipeline mode ("Equation 1 is bypassed, a pluggable estimator first picks a model ..., and a dispatcher
 * (round-robin, shortest-queue, or random) places the request within that model's replica pool").  The model choice is
 * the caller's (the paper's model-picking estimators are comparison systems, out of scope); the library places each
 * request, in input order, inside the chosen tier's replica pool and applies the greedy pass's dead-reckoning update.
 *   model       [host|device] B int32: tier chosen for each request, in [0,M)
 *   outlen      [host|device] B x M fp32 predicted output lengths, or NULL: no dead-reckoning update
 *   policy      0 round-robin (instances of the tier in index order; one cursor per tier, kept across calls),
 *               1 shortest queue (smallest queued_tokens, ties -> smaller index),
 *               2 random (member splitmix64(seed + n) mod pool size, n = requests placed so far on this context)
 *   commit      0: leave the state, cursors and draw counter untouched
 *   assignment  [host|device] B int32; -1 for a request whose tier has no instance
 * Cursors and the draw counter are reset by rb_set_instances. */
rb_status rb_dispatch_pipeline(rb_ctx* ctx, const int32_t* model, const float* outlen, int32_t B, int32_t policy,
                               uint64_t seed, int32_t commit, int32_t* assignment);

/* Batch-level matching replay ("A batch-level matching (e.g. Hungarian) would differ only through within-batch
 * state updates, and an offline replay over the logged score matrices changes 15.6% of assignments").  Finds the
 * assignment a of the B requests that maximises sum_r scores0[r, a(r)] with at most quota[i] requests on instance i and
 * none on an instance filtered out for the request (score -inf) -- the Hungarian method in shortest-augmenting-path form
 * on the transportation problem, fp64 duals, one CTA -- and counts the requests it places differently from `greedy`.
 * The paper does not say how its replay bounds an instance's share of a batch: the quota is the caller's (DESIGN.md
 * reading 26); quota[i] >= B for all i makes the optimum the row-wise argmax.  An offline tool, not on the decision path.
 *   scores0     [host|device] B x I fp32: the batch-start score matrix (rb_decide_from_predictions' scores0)
 *   quota       [host|device] I int32 >= 0
 *   greedy      [host|device] B int32 or NULL: assignment to compare with
 *   match       [host|device] B int32: the optimal assignment (one of them, if several tie)
 *   objective   [host] or NULL: sum of the chosen scores (fp64);   n_diverged [host] or NULL: #{r : match[r] != greedy[r]}
 * 1 <= B <= 4096.  RB_EINVAL when no feasible assignment exists.  Synchronises the context's stream. */
rb_status rb_match_replay(rb_ctx* ctx, const float* scores0, int32_t B, const int32_t* quota, const int32_t* greedy,
                          int32_t* match, double* objective, int32_t* n_diverged);

/* The estimate stage alone (KNN scan + merge + aggregate); outputs as in rb_decide, any may be NULL. */
rb_status rb_estimate(rb_ctx* ctx, const float* query_emb, int32_t B, float* pred_quality,
                      float* pred_outlen, int32_t* nn_idx, float* nn_sim);

/* Number of kernel launches (graph nodes count individually) issued by this context so far. */
int64_t rb_launch_count(const rb_ctx* ctx);

/* Blocks until all work issued on the context's stream has finished. */
rb_status rb_sync(rb_ctx* ctx);

/* Human-readable description of the last failure on ctx ("" if none).  Valid until the next call. */
const char* rb_last_error(const rb_ctx* ctx);

/* Frees everything the context owns.  NULL is allowed. */
void rb_destroy(rb_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* ROUTEBALANCE_H_ */
