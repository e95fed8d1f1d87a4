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
constexpr int kBoxN = 64;          // bank rows per TMA box; slabs are multiples of this
constexpr int kTileK = 64;         // bf16 per K chunk = one 128-byte swizzle row

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
};

// Per-call parameters that change between graph replays live in device memory.
struct CallParams {
  float w_qual, w_lat, w_cost;
  int32_t commit;
};

// ---- launchers (each returns the cudaError of its launch) ---------------------------------------------
// a0: fp32 queries -> bf16 staging [Bpad x d], rows >= B zeroed.
cudaError_t launch_stage_queries(const float* q, __nv_bfloat16* qs, int B, int Bpad, int d, cudaStream_t s);

// a1 (bf16): tcgen05 scan.  part_* are [grid][KCAP][Bpad] (sim fp32 / idx int32, idx -1 = empty).
// Returns the grid size used through *grid_out.  kcap in {16,32,64}.
cudaError_t launch_scan_tc(const CUtensorMap* tm_q, const CUtensorMap* tm_bank, int64_t N, int d, int B, int Bpad,
                           int kcap, int max_grid, float* part_sim, int32_t* part_idx, int* grid_out,
                           cudaStream_t s);
size_t scan_tc_smem_bytes();
cudaError_t scan_tc_prepare();  // opt in to the dynamic shared memory size; call once

// a1 (fp32 storage): exact fp64-accumulated similarities of queries [r0, r0+nq) to sims [nq x N],
// then per-query selection of the kc best (sim desc, idx asc) into cand_* [B x kc].
cudaError_t launch_scan_f32(const float* bank, const float* q, int64_t N, int d, int nq, float* sims, cudaStream_t s);
cudaError_t launch_select_f32(const float* sims, int64_t N, int nq, int kc, float* cand_sim, int32_t* cand_idx,
                              cudaStream_t s);

// a2: merge the per-CTA partial lists into cand_* [B x kc], best first.
cudaError_t launch_merge(const float* part_sim, const int32_t* part_idx, int grid, int kcap, int Bpad, int B, int kc,
                         int64_t N, float* cand_sim, int32_t* cand_idx, cudaStream_t s);

// a3: optional exact re-rank of the kc candidates (bf16 storage), keep k, distance weights, label gather.
cudaError_t launch_aggregate(const __nv_bfloat16* bank, const __nv_bfloat16* qs, int d, int rerank, const float* cand_sim,
                             const int32_t* cand_idx, int kc, int k, const float* bank_quality, const float* bank_outlen,
                             int M, int weight_mode, float eps, int B, int32_t* nn_idx, float* nn_sim, float* pred_q,
                             float* pred_l, cudaStream_t s);

// a4+a5: per-(request, tier) terms, LPT keys, batch-start score matrix.
cudaError_t launch_score(InstTable t, const float* dq, const int32_t* bq, const float* pred_q, const float* pred_l,
                         const int32_t* plen, const CallParams* cp, int B, float* termA, float* termP, float* key,
                         float* scores0, cudaStream_t s);

// a6+a7: LPT sort + greedy dispatch with dead-reckoned updates (single CTA).
cudaError_t launch_dispatch(InstTable t, float* dq, int32_t* bq, const float* pred_l, const float* termA,
                            const float* termP, const float* key, const CallParams* cp, int B, int lpt_enabled,
                            int update_enabled, int32_t* order, int32_t* assignment, float* scores, cudaStream_t s);

// a8: dead reckoning between batches.
cudaError_t launch_advance(InstTable t, float* dq, int32_t* bq, float elapsed_ms, cudaStream_t s);

}  // namespace rb
