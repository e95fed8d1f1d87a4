// orc.cpp -- ORACLE.  Test infrastructure, not product code.
//
// A plain, slow, obviously-correct CPU statement of RouteBalance's per-batch scheduling decision, written
// from the paper text alone (P:Lnnn = line nnn of PAPER.md).  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load this file.  It shares no code, header, table or
// helper with the CUDA library under paper_2606_17949_b200/, and neither includes the other.
//
// The method is a heuristic pipeline (approximate predictor + greedy assignment), so apart from the
// neighbour search -- which is the brute-force definition of "k nearest" -- the oracle follows the
// algorithm step by step, in the paper's order.  Every fp32 line below is ONE IEEE-754 binary32
// round-to-nearest-even operation (build with -ffp-contract=off, no -ffast-math), because the LPT
// assignment must be reproducible bit for bit.  Readings of points where the paper is silent are numbered
// as in DESIGN.md "Readings".
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): hand-worked examples W0/W1/W2 (tests/golden/),
// the 6x-cheaper closed form of P:L90, simplex corners, k=N -> bank mean, k=1 -> nearest row's labels,
// scikit-learn KNeighborsRegressor(weights='distance', algorithm='brute'), single-instance cluster,
// LPT ordering invariant, exhaustive assignment on tiny inputs, price/latency scale invariance,
// tier-loss == masking, advance closed form.  Parity unpinned: none of the functions below; the paper's
// end-to-end outcomes (tier shares, DeepEval quality) need its dataset and cluster and are not computed here.
//
// C ABI, host pointers only, stateless: every function maps input arrays to output arrays.

#include <algorithm>
#include <cmath>
#include <climits>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// bfloat16 = upper 16 bits of binary32.  Round-to-nearest-even from binary32 (reading 4: the storage
// precision of bank and queries is part of the definition).
inline uint16_t f32_to_bf16_rne(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x0040u);  // NaN stays NaN
  uint32_t lsb = (u >> 16) & 1u;
  u += 0x7fffu + lsb;
  return (uint16_t)(u >> 16);
}
inline float bf16_to_f32(uint16_t h) {
  uint32_t u = (uint32_t)h << 16;
  float f;
  std::memcpy(&f, &u, 4);
  return f;
}

// Value of element (row n, column c) of a matrix held as fp32 (dtype 0) or raw bf16 (dtype 1), after
// rounding to the storage dtype `store` (0 = keep fp32, 1 = bf16).
inline double stored_value(const void* base, int dtype, int store, int64_t off) {
  if (dtype == 1) return (double)bf16_to_f32(((const uint16_t*)base)[off]);
  float f = ((const float*)base)[off];
  if (store == 1) f = bf16_to_f32(f32_to_bf16_rne(f));
  return (double)f;
}

}  // namespace

extern "C" {

// Threads the neighbour search uses (reported by bench.py's cpu_baseline as "cores"); no arithmetic.
int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// Sets the thread count of the neighbour search (bench.py's 1-thread figure); no arithmetic.
int orc_set_num_threads(int n) {
#ifdef _OPENMP
  if (n >= 1) omp_set_num_threads(n);
#endif
  (void)n;
  return 0;
}

// Rounds n fp32 values to bf16 (RNE); out receives the raw 16-bit patterns.
int orc_round_bf16(const float* in, uint16_t* out, int64_t n) {
  for (int64_t i = 0; i < n; ++i) out[i] = f32_to_bf16_rne(in[i]);
  return 0;
}

// Step 1-3 ("queries a distance-weighted FAISS KNN index (k=10)"; reading 1: exact inner-product
// search over the stored vectors; reading 3: equal similarities -> smaller bank index first).
//   s[r,n] = fl32( sum_{c=0}^{d-1} (double)x~[r,c] * (double)e~[n,c] ), summed in index order in fp64.
//   nn[r][0..k-1] = the k rows with the largest s, ordered by (s descending, n ascending).
// bank: N x d in bank_dtype (0 fp32 / 1 raw bf16); query: B x d fp32; both rounded to store_dtype first.
int orc_knn(const void* bank, int bank_dtype, int store_dtype, const float* query, int64_t N, int d,
            int B, int k, int32_t* nn_idx, float* nn_sim) {
  if (k < 1 || k > N) return 1;
  std::vector<double> x(d);
  std::vector<float> s(N);
  std::vector<int32_t> ord(N);
  for (int r = 0; r < B; ++r) {
    for (int c = 0; c < d; ++c) x[c] = stored_value(query, 0, store_dtype, (int64_t)r * d + c);
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; ++n) {
      double acc = 0.0;
      for (int c = 0; c < d; ++c) acc += x[c] * stored_value(bank, bank_dtype, store_dtype, n * d + c);
      s[n] = (float)acc;
    }
    std::iota(ord.begin(), ord.end(), 0);
    std::partial_sort(ord.begin(), ord.begin() + k, ord.end(), [&](int32_t a, int32_t b) {
      if (s[a] != s[b]) return s[a] > s[b];
      return a < b;
    });
    for (int j = 0; j < k; ++j) {
      nn_idx[(int64_t)r * k + j] = ord[j];
      nn_sim[(int64_t)r * k + j] = s[ord[j]];
    }
  }
  return 0;
}

// Step 4-5 ("distance-weighted"; "one lookup returns a predicted quality and expected length for
// every candidate").  Reading 2: dist = sqrt(max(0, 2 - 2 s)) (Euclidean distance of unit vectors),
// w = 1/(dist + eps); weight_mode 1 = uniform.  Reading 8: L^ uses the same weights as Q^.
int orc_aggregate(const int32_t* nn_idx, const float* nn_sim, const float* bank_quality,
                  const float* bank_outlen, int B, int k, int M, int weight_mode, float eps,
                  float* pred_quality, float* pred_outlen) {
  std::vector<float> w(k);
  for (int r = 0; r < B; ++r) {
    for (int j = 0; j < k; ++j) {
      if (weight_mode == 1) {
        w[j] = 1.0f;
      } else {
        float t = 2.0f * nn_sim[(int64_t)r * k + j];
        float u = 2.0f - t;
        u = std::max(u, 0.0f);
        float dist = std::sqrt(u);
        float den = dist + eps;
        w[j] = 1.0f / den;
      }
    }
    for (int m = 0; m < M; ++m) {
      float numq = 0.0f, numl = 0.0f, den = 0.0f;
      for (int j = 0; j < k; ++j) {
        int64_t n = nn_idx[(int64_t)r * k + j];
        float pq = w[j] * bank_quality[n * M + m];
        numq = numq + pq;
        float pl = w[j] * bank_outlen[n * M + m];
        numl = numl + pl;
        den = den + w[j];
      }
      pred_quality[(int64_t)r * M + m] = numq / den;
      pred_outlen[(int64_t)r * M + m] = numl / den;
    }
  }
  return 0;
}

// Gradient-boosted TPOT head ("For each (model, GPU) tier we train one XGBoost TPOT head"; P:L131 telemetry:
// "queue depth, pending decode work, active sequences, KV-cache pressure, recent service rate").  The paper's trained
// boosters are not available, so the forest is an INPUT; what is restated here is the evaluation rule of an XGBoost
// regression forest (reading 9b):
//   features of instance i:  x[0] = (float)b_i (active sequences), x[1] = d_i (pending decode work),
//                            x[2+j] = aux[i, j], the remaining telemetry fields, constant during a batch
//   node: feature >= 0 -> internal, go to `left` if x[feature] < value else to `right`; feature < 0 -> leaf `value`
//   prediction of tier t:    p = base[t]; for each tree of the tier, in order: p = p + leaf(tree, x)   (fp32)
//   tpot_i = max(p, 1e-6)   (a TPOT is positive; the floor keeps T^ and the drain rule finite for any forest)
struct orc_forest {
  const int32_t* node_feature;
  const float* node_value;
  const int32_t* node_left;
  const int32_t* node_right;
  const int32_t* tree_root;        // [n_trees] index of each tree's root node
  const int32_t* tier_tree_begin;  // [M+1] trees of tier t: tree_root[tier_tree_begin[t] .. tier_tree_begin[t+1])
  const float* base;               // [M]
  int32_t n_features;              // F = 2 + Fa
  const float* aux;                // [I x Fa] or NULL when Fa = 0
};

static float gbdt_tpot(const orc_forest* f, int t, int32_t b, float d, int i) {
  const int Fa = f->n_features - 2;
  float p = f->base[t];
  for (int tr = f->tier_tree_begin[t]; tr < f->tier_tree_begin[t + 1]; ++tr) {
    int n = f->tree_root[tr];
    while (f->node_feature[n] >= 0) {
      int c = f->node_feature[n];
      float x = (c == 0) ? (float)b : (c == 1) ? d : f->aux[(int64_t)i * Fa + (c - 2)];
      n = (x < f->node_value[n]) ? f->node_left[n] : f->node_right[n];
    }
    p = p + f->node_value[n];
  }
  return std::max(p, 1e-6f);
}

// One row of Eq. 1 for request r against the state (dq, bq).
//   P:L92-95 Eq. 2   C[r,i] = l_r * c_in[m(i)] + L^[r,m(i)] * c_out[m(i)]; "a pre-scoring filter keeps only candidates
//                    whose predicted total cost ... fits within" the request's budget: J_r = {i : C[r,i] <= b_r}.
//                    Reading 24 (the paper is silent on an empty J_r): then J_r = {i : C[r,i] = min_j C[r,j]}, the
//                    cheapest candidates.  No budget (has_budget = 0) or b_r = +inf: J_r = all instances.
//   P:L119           T[r,i] = tpot_i * (d_i/b_i + L^[r,m(i)]); "if the instance has a free decode slot only
//                    the second term applies" (reading 11: free <=> b_i < cap_i); reading 9: linear head
//                    tpot_i = dec*(1+slope*b_i); reading 10: plus a prefill term pre*l_r (pre = 0 -> paper).
//                    latency_mode 1 (P:L227 arm 4, "static per-tier prior (nominal TPOT x predicted length; zero
//                    telemetry)"): T[r,i] = dec[m(i)] * L^[r,m(i)].
//                    latency_mode 2: tpot_i from the tier's gradient-boosted head (gbdt_tpot above) instead of the
//                    linear stand-in; the rest of the formula is unchanged.
//   P:L82-90 Eq. 1   S = w_qual*Q^ + w_cost*(1 - C/max_j C) + w_lat*(1 - T/max_j T), maxima over the
//                    request's candidates j in J_r (reading 13), a zero maximum makes the term 0 (reading 14);
//                    summed in Eq. 1's order (reading 15): (w_q*Q + w_c*cost) + w_l*lat.
//                    Instances outside J_r get S = -inf (they are never chosen).
static void score_row(int I, int M, const int32_t* tier, const int32_t* cap, const float* price_in,
                      const float* price_out, const float* pre, const float* dec, const float* slope,
                      const float* dq, const int32_t* bq, const float* Q, const float* L, int32_t ell,
                      const float* w /*qual,lat,cost*/, int has_budget, float budget, int latency_mode,
                      const orc_forest* forest, float* S, float* T_out /*I or NULL*/, char* cand_out /*I or NULL*/) {
  (void)M;
  std::vector<float> C(I), T(I);
  std::vector<char> cand(I, 1);
  for (int i = 0; i < I; ++i) {
    int t = tier[i];
    float c1 = (float)ell * price_in[t];
    float c2 = L[t] * price_out[t];
    C[i] = c1 + c2;
    if (latency_mode == 1) {
      T[i] = dec[t] * L[t];
    } else {
      float tpot;
      if (latency_mode == 2) {   // reading 9b: the tier's boosted TPOT head over the instance's telemetry
        tpot = gbdt_tpot(forest, t, bq[i], dq[i], i);
      } else {
        float a = slope[t] * (float)bq[i];
        a = 1.0f + a;
        tpot = dec[t] * a;
      }
      float wait = (bq[i] < cap[i]) ? 0.0f : dq[i] / (float)bq[i];
      float u = wait + L[t];
      float v = tpot * u;
      float p = pre[t] * (float)ell;
      T[i] = p + v;
    }
  }
  if (has_budget) {
    bool any = false;
    for (int i = 0; i < I; ++i) {
      cand[i] = (C[i] <= budget) ? 1 : 0;
      any = any || cand[i];
    }
    if (!any) {
      float Cmin = C[0];
      for (int i = 1; i < I; ++i) Cmin = std::min(Cmin, C[i]);
      for (int i = 0; i < I; ++i) cand[i] = (C[i] == Cmin) ? 1 : 0;
    }
  }
  float Cmax = 0.0f, Tmax = 0.0f;
  bool first = true;
  for (int i = 0; i < I; ++i) {
    if (!cand[i]) continue;
    if (first || C[i] > Cmax) Cmax = C[i];
    if (first || T[i] > Tmax) Tmax = T[i];
    first = false;
  }
  for (int i = 0; i < I; ++i) {
    int t = tier[i];
    if (!cand[i]) {
      S[i] = -INFINITY;
    } else {
      float ct = (Cmax > 0.0f) ? 1.0f - (C[i] / Cmax) : 0.0f;
      float lt = (Tmax > 0.0f) ? 1.0f - (T[i] / Tmax) : 0.0f;
      float t1 = w[0] * Q[t];
      float t2 = w[2] * ct;
      float A = t1 + t2;
      float t3 = w[1] * lt;
      S[i] = A + t3;
    }
    if (T_out) T_out[i] = T[i];
    if (cand_out) cand_out[i] = cand[i];
  }
}

// Steps 6-9: Algorithm 1 (caption P:L109, prose P:L111), with the optional pieces of
// SURVEY 8(f) #1 and #2 as arguments whose defaults (budget = NULL, update_mode = 1, tiebreak_mode = 0,
// latency_mode = 0) give the deployed mechanism.
//   key_r = max_m L^[r,m] over tiers that have an instance (reading 16/23), requests dispatched by
//   (key descending, r ascending) when lpt_enabled, else in input order.
//   Each dispatch: S[r,:] from the CURRENT local state; i* = first candidate in the order
//     tiebreak_mode 0: (S descending, d ascending, i ascending)  -- reading 17, "the scheduler's reactive
//                      shortest-queue tiebreak" (P:L227 arm 2)
//     tiebreak_mode 1: (S descending, T^ ascending, i ascending) -- "a predictive T^-argmin tiebreak" (arm 3);
//   then update_mode 1: d[i*] += L^[r,m(i*)] and the decode batch grows by one while a slot is free
//   (reading 18); update_mode 2: d only (P:L121 literally); update_mode 0: no update.
//   max_tokens[r] ("max_tokens clamped to the remaining budget"): floor((b_r - l_r*c_in)/c_out) at the chosen
//   model's prices, clamped to [0, 2^31-128]; INT32_MAX when r has no finite budget (or c_out = 0 and the input fits).
//   scores0 = S[r,:] of every request from the batch-start state (reading 19).
// dq/bq in: batch-start state; dq_out/bq_out: state after the batch (equal to the input when update_mode = 0).
int orc_dispatch_gbdt(int I, int M, const int32_t* tier, const int32_t* cap, const float* price_in,
                      const float* price_out, const float* pre, const float* dec, const float* slope,
                      const float* dq_in, const int32_t* bq_in, const float* quality, const float* outlen,
                      const int32_t* prompt_len, int B, const float* w, const float* budget /*B or NULL*/,
                      int lpt_enabled, int update_mode, int tiebreak_mode, int latency_mode,
                      const orc_forest* forest /*latency_mode 2*/, int32_t* assignment, float* scores,
                      float* scores0, int32_t* order, int32_t* max_tokens, float* dq_out, int32_t* bq_out) {
  if (latency_mode == 2 && forest == nullptr) return 1;
  std::vector<float> dq(dq_in, dq_in + I);
  std::vector<int32_t> bq(bq_in, bq_in + I);
  std::vector<char> present(M, 0);
  for (int i = 0; i < I; ++i) present[tier[i]] = 1;

  std::vector<float> key(B);
  for (int r = 0; r < B; ++r) {
    bool first = true;
    float kmax = 0.0f;
    for (int m = 0; m < M; ++m) {
      if (!present[m]) continue;
      float l = outlen[(int64_t)r * M + m];
      if (first || l > kmax) kmax = l;
      first = false;
    }
    key[r] = kmax;
  }
  std::vector<int32_t> ord(B);
  std::iota(ord.begin(), ord.end(), 0);
  if (lpt_enabled) {
    std::stable_sort(ord.begin(), ord.end(), [&](int32_t a, int32_t b) { return key[a] > key[b]; });
  }

  std::vector<float> S(I), T(I);
  std::vector<char> cand(I);
  for (int r = 0; r < B; ++r) {
    score_row(I, M, tier, cap, price_in, price_out, pre, dec, slope, dq_in, bq_in, quality + (int64_t)r * M,
              outlen + (int64_t)r * M, prompt_len[r], w, budget != nullptr, budget ? budget[r] : 0.0f, latency_mode,
              forest, S.data(), nullptr, nullptr);
    if (scores0) std::copy(S.begin(), S.end(), scores0 + (int64_t)r * I);
  }

  for (int j = 0; j < B; ++j) {
    int r = ord[j];
    const float* Q = quality + (int64_t)r * M;
    const float* L = outlen + (int64_t)r * M;
    score_row(I, M, tier, cap, price_in, price_out, pre, dec, slope, dq.data(), bq.data(), Q, L, prompt_len[r], w,
              budget != nullptr, budget ? budget[r] : 0.0f, latency_mode, forest, S.data(), T.data(), cand.data());
    int best = -1;
    for (int i = 0; i < I; ++i) {
      if (!cand[i]) continue;
      if (best < 0) { best = i; continue; }
      float ti = tiebreak_mode == 1 ? T[i] : dq[i];
      float tb = tiebreak_mode == 1 ? T[best] : dq[best];
      if (S[i] > S[best] || (S[i] == S[best] && ti < tb)) best = i;
    }
    assignment[r] = best;
    if (scores) std::copy(S.begin(), S.end(), scores + (int64_t)r * I);
    if (order) order[j] = r;
    if (max_tokens) {
      int32_t mt = INT32_MAX;
      if (budget && budget[r] < INFINITY) {
        int t = tier[best];
        float c1 = (float)prompt_len[r] * price_in[t];
        float rem = budget[r] - c1;
        if (price_out[t] > 0.0f) {
          float q = rem / price_out[t];
          q = std::floor(q);
          q = std::max(q, 0.0f);
          q = std::min(q, 2147483520.0f);
          mt = (q == q) ? (int32_t)q : 0;
        } else {
          mt = (rem >= 0.0f) ? INT32_MAX : 0;
        }
      }
      max_tokens[r] = mt;
    }
    if (update_mode != 0) {
      dq[best] = dq[best] + L[tier[best]];
      if (update_mode == 1 && bq[best] < cap[best]) bq[best] += 1;
    }
  }
  if (dq_out) std::copy(dq.begin(), dq.end(), dq_out);
  if (bq_out) std::copy(bq.begin(), bq.end(), bq_out);
  return 0;
}

int orc_dispatch(int I, int M, const int32_t* tier, const int32_t* cap, const float* price_in,
                 const float* price_out, const float* pre, const float* dec, const float* slope,
                 const float* dq_in, const int32_t* bq_in, const float* quality, const float* outlen,
                 const int32_t* prompt_len, int B, const float* w, const float* budget /*B or NULL*/,
                 int lpt_enabled, int update_mode, int tiebreak_mode, int latency_mode, int32_t* assignment,
                 float* scores, float* scores0, int32_t* order, int32_t* max_tokens, float* dq_out,
                 int32_t* bq_out) {
  return orc_dispatch_gbdt(I, M, tier, cap, price_in, price_out, pre, dec, slope, dq_in, bq_in, quality, outlen,
                           prompt_len, B, w, budget, lpt_enabled, update_mode, tiebreak_mode, latency_mode, nullptr,
                           assignment, scores, scores0, order, max_tokens, dq_out, bq_out);
}

// tpot of every instance from the boosted head (what latency_mode 2 uses), for tests of the forest rule alone.
int orc_gbdt_tpot(int I, const int32_t* tier, const orc_forest* forest, const float* dq, const int32_t* bq,
                  float* tpot) {
  for (int i = 0; i < I; ++i) tpot[i] = gbdt_tpot(forest, tier[i], bq[i], dq[i], i);
  return 0;
}

// The deployed mechanism: no budgets, reactive tie-break, live latency, update of d and b.
int orc_decide_from_predictions(int I, int M, const int32_t* tier, const int32_t* cap,
                                const float* price_in, const float* price_out, const float* pre,
                                const float* dec, const float* slope, const float* dq_in,
                                const int32_t* bq_in, const float* quality, const float* outlen,
                                const int32_t* prompt_len, int B, const float* w, int lpt_enabled,
                                int update_enabled, int32_t* assignment, float* scores, float* scores0,
                                int32_t* order, float* dq_out, int32_t* bq_out) {
  return orc_dispatch(I, M, tier, cap, price_in, price_out, pre, dec, slope, dq_in, bq_in, quality, outlen,
                      prompt_len, B, w, nullptr, lpt_enabled, update_enabled ? 1 : 0, 0, 0, assignment, scores,
                      scores0, order, nullptr, dq_out, bq_out);
}

// Step 10 (BASELINE.json rb_advance_state; reading 22: the drain rule is ours, the paper re-reads telemetry):
// each instance with b_i > 0 completes b_i tokens every tpot_i ms.
int orc_advance_state(int I, const int32_t* tier, const float* dec, const float* slope, float elapsed_ms,
                      float* dq, int32_t* bq) {
  for (int i = 0; i < I; ++i) {
    if (bq[i] <= 0) continue;
    int t = tier[i];
    float a = slope[t] * (float)bq[i];
    a = 1.0f + a;
    float tpot = dec[t] * a;
    float q = elapsed_ms / tpot;
    float done = (float)bq[i] * q;
    float d = dq[i] - done;
    d = std::max(d, 0.0f);
    dq[i] = d;
    if (d == 0.0f) bq[i] = 0;
  }
  return 0;
}

// Adaptive batch size ("Batch size is adaptive -- larger when more instances are busy, smaller when idle"; P:L191
// "Adaptive sizing ties t_form to cluster busyness").  The paper gives no rule; reading 27:
//   an instance is busy  <=>  it has no free decode slot, b_i >= cap_i (the condition under which the wait term of
//                             P:L119 applies, reading 11);
//   n_busy = #{i : b_i >= cap_i};
//   target = bs_min + floor((bs_max - bs_min) * n_busy / I)          (integers)
// so that an idle cluster gives bs_min, a saturated one bs_max, and bs_min = bs_max is the ablation's fixed batch size
// ("adaptive-off", "Fixed batch size ... bs=1 / 16 / 32").
int orc_batch_target(int I, const int32_t* cap, const int32_t* bq, int bs_min, int bs_max, int32_t* target,
                     int32_t* n_busy) {
  if (I < 1 || bs_min < 1 || bs_max < bs_min) return 1;
  int busy = 0;
  for (int i = 0; i < I; ++i)
    if (bq[i] >= cap[i]) busy += 1;
  *target = (int32_t)(bs_min + ((int64_t)(bs_max - bs_min) * busy) / I);
  if (n_busy) *n_busy = busy;
  return 0;
}

// Step 10 with the boosted head: the same drain rule, tpot_i from gbdt_tpot.
int orc_advance_state_gbdt(int I, const int32_t* tier, const orc_forest* forest, float elapsed_ms, float* dq,
                           int32_t* bq) {
  for (int i = 0; i < I; ++i) {
    if (bq[i] <= 0) continue;
    float tpot = gbdt_tpot(forest, tier[i], bq[i], dq[i], i);
    float q = elapsed_ms / tpot;
    float done = (float)bq[i] * q;
    float d = dq[i] - done;
    d = std::max(d, 0.0f);
    dq[i] = d;
    if (d == 0.0f) bq[i] = 0;
  }
  return 0;
}

// A second, separately labelled CPU figure for bench.py only (never used for parity): the same brute-force
// scan with an fp32 accumulator whose sum the compiler may reorder and vectorise (omp simd reduction; AVX2 when the
// host has it).  Returns the index of the best row per query.
#define ORC_FAST_SCAN_BODY                                              \
  for (int r = 0; r < B; ++r) {                                         \
    float bs = -INFINITY;                                               \
    int32_t bi = 0;                                                     \
    const float* x = query + (int64_t)r * d;                            \
    for (int64_t n = 0; n < N; ++n) {                                   \
      const float* e = bank + n * d;                                    \
      float acc = 0.0f;                                                 \
      _Pragma("omp simd reduction(+ : acc)")                            \
      for (int c = 0; c < d; ++c) acc += x[c] * e[c];                   \
      if (acc > bs) { bs = acc; bi = (int32_t)n; }                      \
    }                                                                   \
    best[r] = bi;                                                       \
  }
}  // extern "C"
__attribute__((target("avx2"))) static void scan_fast_avx2(const float* bank, const float* query, int64_t N, int d, int B,
                                                           int32_t* best) {
  ORC_FAST_SCAN_BODY
}
static void scan_fast_base(const float* bank, const float* query, int64_t N, int d, int B, int32_t* best) {
  ORC_FAST_SCAN_BODY
}
extern "C" {
int orc_scan_fast_f32(const float* bank, const float* query, int64_t N, int d, int B, int32_t* best) {
  if (__builtin_cpu_supports("avx2")) scan_fast_avx2(bank, query, N, d, B, best);
  else scan_fast_base(bank, query, N, d, B, best);
  return 0;
}

}  // extern "C"

// ---- pipeline mode: "Equation 1 is bypassed, a pluggable estimator first picks a model ..., and a dispatcher
// (round-robin, shortest-queue, or random) places the request within that model's replica pool."  The model choice is an
// INPUT here (the paper's model-picking estimators are comparison systems); what is stated is the three dispatchers,
// in input order, over the same dead-reckoned state and with the same update as the greedy pass (reading 18):
//   policy 0 round-robin    the tier's instances in index order, a cursor per tier that persists across batches
//   policy 1 shortest queue  the tier's instance with the smallest d_i, ties -> smaller i
//   policy 2 random          member (splitmix64(seed + counter) mod n_m) of the tier's instances in index order; counter =
//                            number of requests placed so far (persists across batches), so both sides draw the same numbers
// A request whose tier has no instance gets assignment -1 and changes nothing.
extern "C" {

static inline uint64_t splitmix64(uint64_t x) {
  x += 0x9e3779b97f4a7c15ull;
  x = (x ^ (x >> 30)) * 0xbf58476d1ce4e5b9ull;
  x = (x ^ (x >> 27)) * 0x94d049bb133111ebull;
  return x ^ (x >> 31);
}

uint64_t orc_splitmix64(uint64_t x) { return splitmix64(x); }

int orc_pipeline_dispatch(int I, int M, const int32_t* tier, const int32_t* cap, const float* dq_in, const int32_t* bq_in,
                          const int32_t* model, const float* outlen /*B x M or NULL: no update*/, int B, int policy,
                          uint64_t seed, uint64_t* counter /*in/out*/, int32_t* cursor /*M, in/out*/, int32_t* assignment,
                          float* dq_out, int32_t* bq_out) {
  std::vector<float> dq(dq_in, dq_in + I);
  std::vector<int32_t> bq(bq_in, bq_in + I);
  for (int r = 0; r < B; ++r) {
    const int m = model[r];
    std::vector<int> members;
    if (m >= 0 && m < M)
      for (int i = 0; i < I; ++i)
        if (tier[i] == m) members.push_back(i);
    if (members.empty()) { assignment[r] = -1; continue; }
    const int n = (int)members.size();
    int pick;
    if (policy == 0) {
      pick = members[cursor[m] % n];
      cursor[m] = (cursor[m] + 1) % n;
    } else if (policy == 1) {
      pick = members[0];
      for (int i : members)
        if (dq[i] < dq[pick]) pick = i;
    } else {
      pick = members[(int)(splitmix64(seed + *counter) % (uint64_t)n)];
    }
    *counter += 1;
    assignment[r] = pick;
    if (outlen) {
      dq[pick] = dq[pick] + outlen[(int64_t)r * M + m];
      if (bq[pick] < cap[pick]) bq[pick] += 1;
    }
  }
  if (dq_out) std::copy(dq.begin(), dq.end(), dq_out);
  if (bq_out) std::copy(bq.begin(), bq.end(), bq_out);
  return 0;
}

}  // extern "C"
