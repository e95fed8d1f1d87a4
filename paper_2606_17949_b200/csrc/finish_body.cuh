// finish_body.cuh -- steps a2 + a3 + a4 for ONE query by one CTA: cross-CTA top-k merge of the scan's partial lists,
// exact re-rank, distance-weighted aggregate and the per-(request, tier) score terms (Eq. 1 / Eq. 2).
// A device function so that the standalone finishing kernel (estimate.cu) and the tail of the fused decision kernel
// (scan_tc.cu) run the same code.  Product code; included by those two files only.
//
// The work is a chain of short dependent phases executed once (latency-bound: a few hundred instructions of one warp
// cost a microsecond), so every phase is spread over the lanes and warps of the CTA, loops stay rolled, and the rare
// cases live in functions that are not inlined.
//  load    the query's partial lists (sorted by key, descending) become 64-bit keys in shared memory.
//  bound   the threads form groups of kGroupLanes lanes; the kc-th largest group maximum is reached by kc distinct
//          entries, so every member of the kc best reaches it too (admission bound).
//  select  entries at or above the bound (a few dozen) are compacted and ranked by counting (keys are distinct);
//          more survivors than slots (equal similarities, a bank sorted by topic): kc rounds of a block-wide maximum.
//  rescan  the scan may keep fewer entries per (CTA, query) than kc (short lists make its warm-up cheap).  A list
//          whose last entry made the kc best may hide further members; the bank rows of such a slab (rare: several of
//          a query's kc best in one of ~148 slabs) are searched again here, exactly, and the selection is redone over
//          the other slabs' candidates and the slab's own best.
//  re-rank (bf16 storage): the kc candidates' similarities are recomputed from the stored bf16 rows with fp64
//          accumulation (products of bf16 values are exact), rounded once to fp32, re-ordered by
//          (s desc, n asc); the best k are the neighbours.
//  aggregate:
//          t = 2*s; u = 2 - t; u = max(u,0); dist = sqrt(u); w = 1/(dist + eps)      (uniform mode: w = 1)
//          num_m = sum_j w_j*label[n_j,m] (j ascending, multiply then add); den = sum_j w_j; pred = num/den
//  terms   (with_terms; Eq. 2, Eq. 1):
//          c1 = (float)l*pin; c2 = L*pout; C = c1 + c2; Cmax over tiers that have an instance;
//          ct = Cmax > 0 ? 1 - C/Cmax : 0; A = wq*Q + wc*ct; P = pre*(float)l; key = max_m L
#pragma once
#include "rb_internal.cuh"

namespace rb {
namespace {

constexpr int kFinThreadsMax = 768;                // (a block of 768 threads may use 85 registers per thread)
constexpr int kFinWarpsMax = kFinThreadsMax / 32;
constexpr int kMaxFlag = 16;                      // flagged lists per query <= kc / kcap
constexpr int kSurvMax = 256;                     // survivors of the admission bound that are ranked by counting
constexpr int kRescanKeep = 64;                   // entries every warp keeps of a slab it searches again (>= kMaxK)

// Total order of candidates: similarity descending, bank index ascending (reading 3), as one 64-bit key whose
// unsigned order is that order (larger key = better).  Key 0 is below every real candidate.
__device__ __forceinline__ unsigned long long fin_key(float sim, int32_t idx) {
  return ((unsigned long long)rb_f2o(sim) << 32) | (unsigned long long)(0xffffffffu - (uint32_t)idx);
}

// Shared-memory scratch of one finishing CTA (besides the keys of the lists themselves).
struct FinScratch {
  uint32_t red[2][kFinWarpsMax][2];
  uint32_t gmax[kFinThreadsMax];
  unsigned long long surv[kSurvMax];
  unsigned long long cand[kMaxK];
  float w[kMaxK];
  float lab[kMaxK][2 * kMaxM];    // w_c * label of the kc candidates: [quality(M) | outlen(M)]
  float prod[kMaxK][2 * kMaxM];   // the same rows by final rank
  unsigned long long ckey[kMaxK]; // exact keys of the candidates
  float wr[kMaxK];                // weights by final rank
  float Q[kMaxM], L[kMaxM];
  int flag[kMaxFlag];
  int nsurv, nflag;
  uint32_t tau;
};

// s = fl32( sum_c (double)x[c]*(double)e[c] ) of two bf16 rows (nvec uint4 of 8 values each, nvec <= 128), the 32
// lanes' fp64 partials added by shuffles.  All of a lane's loads are issued before the first product.
__device__ __forceinline__ float exact_sim_bf16(const uint4* __restrict__ qrow, const uint4* __restrict__ brow, int nvec,
                                                int lane) {
  double acc = 0.0;
#pragma unroll 1
  for (int v0 = lane; v0 < nvec; v0 += 128) {
    uint4 xb[4], eb[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int v = v0 + 32 * u;
      if (v < nvec) { xb[u] = qrow[v]; eb[u] = __ldg(brow + v); }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (v0 + 32 * u < nvec) {
        const __nv_bfloat162* xp = reinterpret_cast<const __nv_bfloat162*>(&xb[u]);
        const __nv_bfloat162* ep = reinterpret_cast<const __nv_bfloat162*>(&eb[u]);
#pragma unroll
        for (int h = 0; h < 4; ++h) {
          const float2 xf = __bfloat1622float2(xp[h]), ef = __bfloat1622float2(ep[h]);
          acc = fma((double)xf.x, (double)ef.x, acc);
          acc = fma((double)xf.y, (double)ef.y, acc);
        }
      }
    }
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  return (float)acc;
}

// s = fl32( sum_c (double)x[c]*(double)e[c] ) of two fp32 rows of d values (d % 4 == 0), lanes' fp64 partials added by shuffles.
__device__ __forceinline__ float exact_sim_f32(const float4* __restrict__ qrow, const float4* __restrict__ brow, int nvec4,
                                               int lane) {
  double acc = 0.0;
#pragma unroll 2
  for (int v = lane; v < nvec4; v += 32) {
    const float4 x = qrow[v], e = __ldg(brow + v);
    acc = fma((double)x.x, (double)e.x, acc);
    acc = fma((double)x.y, (double)e.y, acc);
    acc = fma((double)x.z, (double)e.z, acc);
    acc = fma((double)x.w, (double)e.w, acc);
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  return (float)acc;
}
// Exact similarity of query row r to bank row n in the storage precision (a.rerank: 1 bf16 rows, 2 fp32 rows).
__device__ __forceinline__ float exact_sim(const FinishArgs& a, const float* __restrict__ q32, int r, int64_t n, int lane) {
  if (a.rerank == 2)
    return exact_sim_f32(reinterpret_cast<const float4*>(q32 + (size_t)r * a.d),
                         reinterpret_cast<const float4*>(a.bank32 + (size_t)n * a.d), a.d / 4, lane);
  return exact_sim_bf16(reinterpret_cast<const uint4*>(a.qs + (size_t)r * a.d),
                        reinterpret_cast<const uint4*>(a.bank + (size_t)n * a.d), a.d / 8, lane);
}

// kc rounds of a block-wide maximum over distinct 64-bit keys: each round takes the largest key below the previous
// pick (keys [n] in shared memory; 0 = empty).  Result in out[0..kc), descending (0 = exhausted).  All threads of the
// block must call.  Rare path: kept out of line.
__device__ __noinline__ void block_select_topk(const unsigned long long* keys, int n, int kc,
                                               uint32_t (*s_red)[kFinWarpsMax][2], unsigned long long* out) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nwarps = blockDim.x >> 5;
  unsigned long long prev = ~0ull;
#pragma unroll 1
  for (int j = 0; j < kc; ++j) {
    unsigned long long best = 0ull;
    for (int e = tid; e < n; e += blockDim.x) {
      const unsigned long long key = keys[e];
      if (key < prev && key > best) best = key;
    }
    const uint32_t hi = (uint32_t)(best >> 32), lo = (uint32_t)best;
    const uint32_t whi = __reduce_max_sync(0xffffffffu, hi);
    const uint32_t wlo = __reduce_max_sync(0xffffffffu, hi == whi ? lo : 0u);
    if (lane == 0) { s_red[j & 1][warp][0] = whi; s_red[j & 1][warp][1] = wlo; }
    __syncthreads();
    const uint32_t xhi = lane < nwarps ? s_red[j & 1][lane][0] : 0u;
    const uint32_t xlo = lane < nwarps ? s_red[j & 1][lane][1] : 0u;
    const uint32_t ghi = __reduce_max_sync(0xffffffffu, xhi);
    const uint32_t glo = __reduce_max_sync(0xffffffffu, xhi == ghi ? xlo : 0u);
    prev = ((unsigned long long)ghi << 32) | glo;
    if (tid == 0) out[j] = prev;
    if (prev == 0ull) prev = 1ull;   // exhausted: later rounds find nothing (key 0 is below every real candidate)
  }
  __syncthreads();
}

// Rows [row0, row1) of slab c (the scan's split of the bank: slab c = units [units*c/nslabs, units*(c+1)/nslabs)).
__device__ __forceinline__ void slab_rows(const FinishArgs& a, int c, int nslabs, int64_t* row0, int64_t* row1) {
  const int64_t units = (a.N + a.slab_unit - 1) / a.slab_unit;
  *row0 = units * c / nslabs * a.slab_unit;
  int64_t r1 = units * (c + 1) / nslabs * a.slab_unit;
  *row1 = r1 > a.N ? a.N : r1;
}

// The slabs whose list may hide members of the kc best (last entry at or above kstar, the kc-th best key found) are
// searched again with exact similarities; S.cand becomes the kc best of those slabs' rows and of the candidates that
// came from the other slabs.  s_keys is overwritten ([nwarps][kRescanKeep] + [kc]).  All threads must call; rare path.
__device__ __noinline__ void rescan_slabs(const FinishArgs a, const float* q32, int r, unsigned long long kstar,
                                          unsigned long long* s_keys, FinScratch& S) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nwarps = blockDim.x >> 5;
  const int kc = a.kc, kcap = a.kcap;
  if (tid == 0) S.nflag = 0;
  __syncthreads();
  for (int l = tid; l < a.nlists; l += blockDim.x) {
    const unsigned long long last = s_keys[(size_t)l * kcap + kcap - 1];
    if (last != 0ull && last >= kstar) {
      const int p = atomicAdd(&S.nflag, 1);
      if (p < kMaxFlag) S.flag[p] = l / a.lists_per_cta;
    }
  }
  __syncthreads();
  if (tid == 0) {   // lists -> slabs, each once
    const int nl = min(S.nflag, kMaxFlag);
    int nc = 0;
    for (int f = 0; f < nl; ++f) {
      const int c = S.flag[f];
      bool seen = false;
      for (int g = 0; g < nc; ++g) seen |= (S.flag[g] == c);
      if (!seen) S.flag[nc++] = c;
    }
    S.nflag = nc;
  }
  __syncthreads();
  const int nflag = S.nflag;
  const int nslabs = a.nlists / a.lists_per_cta;
  // every warp keeps the best 64 of the rows it visits: rank l in lane l (la) and rank 32 + l (lb)
  unsigned long long la = 0, lb = 0, thr = 0;
  for (int f = 0; f < nflag; ++f) {
    int64_t row0, row1;
    slab_rows(a, S.flag[f], nslabs, &row0, &row1);
    for (int64_t n = row0 + warp; n < row1; n += nwarps) {
      const float sx = exact_sim(a, q32, r, n, lane);
      const unsigned long long x = fin_key(sx, (int32_t)n);
      if (sx == sx && x > thr) {
        const int p = __popc(__ballot_sync(0xffffffffu, la > x)) + __popc(__ballot_sync(0xffffffffu, lb > x));
        const unsigned long long a_up = __shfl_up_sync(0xffffffffu, la, 1), b_up = __shfl_up_sync(0xffffffffu, lb, 1);
        const unsigned long long a_last = __shfl_sync(0xffffffffu, la, 31);
        const unsigned long long b_prev = (lane == 0) ? a_last : b_up;
        la = (lane < p) ? la : ((lane == p) ? x : a_up);
        lb = (lane + 32 < p) ? lb : ((lane + 32 == p) ? x : b_prev);
        thr = (kc <= 32) ? __shfl_sync(0xffffffffu, la, kc - 1) : __shfl_sync(0xffffffffu, lb, kc - 33);
      }
    }
  }
  __syncthreads();   // everybody is done with the list keys
  s_keys[(size_t)warp * kRescanKeep + lane] = la;
  s_keys[(size_t)warp * kRescanKeep + 32 + lane] = lb;
  if (tid < kc) {    // candidates from the other slabs stay in the running
    const unsigned long long key = S.cand[tid];
    bool from_flagged = false;
    if (key != 0ull) {
      const int64_t n = (int64_t)(0xffffffffu - (uint32_t)key);
      for (int f = 0; f < nflag; ++f) {
        int64_t row0, row1;
        slab_rows(a, S.flag[f], nslabs, &row0, &row1);
        from_flagged |= (n >= row0 && n < row1);
      }
    }
    s_keys[(size_t)nwarps * kRescanKeep + tid] = from_flagged ? 0ull : key;
  }
  __syncthreads();
  block_select_topk(s_keys, nwarps * kRescanKeep + kc, kc, S.red, S.cand);
}

// Dynamic shared memory the keys need: all list entries; the rescan reuses the space for the warps' own lists and the
// other slabs' candidates.
__host__ __device__ inline size_t fin_keys_bytes(int nlists, int kcap) {
  const size_t n1 = (size_t)nlists * kcap * 8;
  const size_t n2 = (size_t)(kFinWarpsMax * kRescanKeep + kMaxK) * 8;
  return n1 > n2 ? n1 : n2;
}

// Steps a2-a4 for query r; every thread of the CTA (blockDim.x a multiple of 32, at least 64, at most kFinThreadsMax)
// must call it, after the lists are visible.  s_keys: fin_keys_bytes() of shared memory, 16-byte aligned; S: scratch.
// On return warp 0 has written the predictions (and terms) of the query; the other warps pass through.
// What the phases are written to (ncu on the C2 workload): the kernel is bound by the NUMBER of warp instructions --
// 19 warps share 4 issue slots and every instruction of a phase that all warps run is paid 19 times -- and by the
// dependent shared-memory / shuffle / vote latencies (20-30 cycles each) between its barriers.
__device__ __forceinline__ void finish_query(const FinishArgs& a, const InstTable& t, const CallParams* __restrict__ cp,
                                             int r, unsigned long long* s_keys, FinScratch& S) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nthreads = blockDim.x, nwarps = blockDim.x >> 5;
  const int kc = a.kc, k = a.k, kcap = a.kcap, M = a.M;
  const int total = a.nlists * kcap;
  // coefficients of the score terms: requested now, consumed at the very end (their latency hides behind the merge)
  float c_pin = 0.0f, c_pout = 0.0f, c_pre = 0.0f, c_ell = 0.0f, c_budget = 0.0f;
  bool has_budget = false;
  int c_present = 0;
  if (a.with_terms && tid < M) {
    c_pin = t.price_in[tid];
    c_pout = t.price_out[tid];
    c_pre = t.pre[tid];
    c_present = t.present[tid];
    c_ell = (float)cp->plen[r];
    has_budget = cp->budget != nullptr;
    if (has_budget) c_budget = cp->budget[r];
  }
  if (tid == 0) { S.nsurv = 0; S.tau = 0u; }
  if (tid < kc) S.cand[tid] = 0ull;

  // ---- load: lists -> keys in shared memory; every thread remembers the best similarity it has seen ----
  uint32_t tmax = 0u;
  const bool quads = a.records != 0;   // query-major records of 4 ready-made keys (scan_tc.cu): one item = one quad
  const int step = quads ? 4 : 1, nitems = quads ? total >> 2 : total;
  if (quads) {
    const uint4* rec = reinterpret_cast<const uint4*>(a.part_sim) + (size_t)r * nitems * 2;
    uint4* dst = reinterpret_cast<uint4*>(s_keys);
#pragma unroll 1
    for (int e = tid; e < nitems; e += nthreads) {
      const uint4 ua = __ldcg(rec + 2 * e), ub = __ldcg(rec + 2 * e + 1);   // (lo, hi) x 4
      dst[2 * e] = ua;
      dst[2 * e + 1] = ub;
      tmax = max(max(tmax, ua.y), max(ua.w, max(ub.y, ub.w)));
    }
  } else {   // [nlists][Bpad][kcap] similarity / index arrays (CTA-pair scan, fp32-storage scan), entry by entry
#pragma unroll 1
    for (int e = tid; e < total; e += nthreads) {
      const int c = e / kcap, j = e - c * kcap;
      const size_t off = ((size_t)c * a.Bpad + r) * kcap + j;
      const int32_t id = __ldcg(a.part_idx + off);
      const unsigned long long key = ((uint32_t)id < (uint32_t)a.N) ? fin_key(__ldcg(a.part_sim + off), id) : 0ull;
      s_keys[e] = key;
      tmax = max(tmax, (uint32_t)(key >> 32));
    }
  }
  // ---- bound: the threads that hold entries form groups of adjacent lanes, as coarse as still leaves 2 kc groups;
  // the kc-th largest group maximum is reached by kc distinct entries, so every member of the kc best reaches it
  // too.  About kc + 6 entries survive.  The groups are ranked by counting: the
  // lanes of a group share its G comparisons and add their counts up by shuffles. ----
  const int nact = min(nthreads, nitems);   // threads that loaded something
  int gshift = 5;   // groups of 2^gshift lanes: the coarsest that still leaves 2 kc groups
  while (gshift > 0 && ((nact + (1 << gshift) - 1) >> gshift) < 2 * kc) --gshift;
  const int glanes = 1 << gshift;
  for (int o = 1; o < glanes; o <<= 1) tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
  const int ngroups = (nact + glanes - 1) >> gshift;   // <= kFinThreadsMax
  const bool bounded = ngroups >= kc && total > kSurvMax;   // (a small input is ranked whole)
  const int g = tid >> gshift;
  if ((tid & (glanes - 1)) == 0 && g < ngroups) S.gmax[g] = tmax;
  __syncthreads();
  if (bounded) {
    int ahead = 0;
    if (g < ngroups) {
#pragma unroll 2
      for (int j = tid & (glanes - 1); j < ngroups; j += glanes) {
        const uint32_t o = S.gmax[j];
        ahead += (o > tmax) || (o == tmax && j < g);
      }
    }
    for (int o = 1; o < glanes; o <<= 1) ahead += __shfl_xor_sync(0xffffffffu, ahead, o);
    if ((tid & (glanes - 1)) == 0 && g < ngroups && ahead == kc - 1) S.tau = tmax;   // ranks are distinct: one writer
    __syncthreads();
  }
  // ---- select: survivors of the bound, compacted (one shared-memory atomic per warp and step; any order) ----
  const uint32_t tau = S.tau;
  bool maybe_hidden = false;   // a list whose LAST entry reaches the bound may be popped completely
#pragma unroll 1
  for (int e0 = 0; e0 < nitems; e0 += nthreads) {   // every thread revisits the entries it wrote itself
    const int e = e0 + tid;
    int c = 0;
    unsigned long long kq[4] = {0ull, 0ull, 0ull, 0ull};
    if (e < nitems) {
#pragma unroll
      for (int h = 0; h < 4; ++h) {
        if (h < step) {
          kq[h] = s_keys[step * e + h];
          c += (kq[h] != 0ull && (uint32_t)(kq[h] >> 32) >= tau);   // sorted within a quad: the survivors are its first c
        }
      }
      if (a.rescan && c == step && ((step * e + step) % kcap) == 0) maybe_hidden = true;
    }
    const uint32_t b0 = __ballot_sync(0xffffffffu, c & 1), b1 = __ballot_sync(0xffffffffu, c & 2),
                   b2 = __ballot_sync(0xffffffffu, c & 4);
    if ((b0 | b1 | b2) == 0u) continue;   // warp-uniform
    const uint32_t lt = (1u << lane) - 1u;
    const int before = __popc(b0 & lt) + 2 * __popc(b1 & lt) + 4 * __popc(b2 & lt);
    int base = 0;
    if (lane == 0) base = atomicAdd(&S.nsurv, __popc(b0) + 2 * __popc(b1) + 4 * __popc(b2));
    base = __shfl_sync(0xffffffffu, base, 0) + before;
#pragma unroll
    for (int h = 0; h < 4; ++h)
      if (h < c && base + h < kSurvMax) S.surv[base + h] = kq[h];
  }
  const int any_hidden = __syncthreads_or(maybe_hidden);
  const int nsurv = S.nsurv;
  if (nsurv <= kSurvMax) {
    // rank by counting (keys are distinct): `sl` adjacent lanes share the comparisons of one survivor
    int sshift = 5;
    while (sshift > 0 && (nsurv << sshift) > nthreads) --sshift;
    const int sl = 1 << sshift;
    const int c = tid >> sshift, s = tid & (sl - 1);
    const unsigned long long mine = c < nsurv ? S.surv[c] : 0ull;
    int ahead = 0;
    if (c < nsurv) {
#pragma unroll 2
      for (int j = s; j < nsurv; j += sl) ahead += S.surv[j] > mine;
    }
    for (int o = 1; o < sl; o <<= 1) ahead += __shfl_xor_sync(0xffffffffu, ahead, o);
    if (s == 0 && c < nsurv && ahead < kc) S.cand[ahead] = mine;
    __syncthreads();
  } else {
    block_select_topk(s_keys, total, kc, S.red, S.cand);
  }
  // ---- rescan of slabs whose list may hide members (only if some list's last entry reached the bound) ----
  if (any_hidden) {
    const unsigned long long kstar = S.cand[kc - 1];
    bool flagged = false;
    for (int l = tid; l < a.nlists; l += nthreads) {
      const unsigned long long last = s_keys[(size_t)l * kcap + kcap - 1];
      flagged |= (last != 0ull && last >= kstar);
    }
    if (__syncthreads_or(flagged)) rescan_slabs(a, a.q32, r, kstar, s_keys, S);
  }

  // ---- exact re-rank: warp c recomputes candidate c, then -- without waiting for the others -- its weight and
  // its weighted labels (neither depends on the candidate's final rank) ----
#pragma unroll 1
  for (int c = warp; c < kc; c += nwarps) {
    const unsigned long long key = S.cand[c];
    const int32_t id = key ? (int32_t)(0xffffffffu - (uint32_t)key) : -1;
    float sx = key ? rb_o2f((uint32_t)(key >> 32)) : -INFINITY;
    float l = 0.0f;   // the labels are requested first: independent of the bank row's loads
    if (id >= 0 && lane < 2 * M)
      l = (lane < M) ? __ldg(a.bank_quality + (size_t)id * M + lane) : __ldg(a.bank_outlen + (size_t)id * M + lane - M);
    if (id >= 0 && a.rerank) sx = exact_sim(a, a.q32, r, id, lane);
    float w = 1.0f;
    if (id < 0) {
      w = 0.0f;   // fewer than kc rows reachable; sorts last and adds +0 if it is ever summed
    } else if (a.weight_mode == 0) {
      const float tt = __fmul_rn(2.0f, sx);
      float u = __fsub_rn(2.0f, tt);
      u = fmaxf(u, 0.0f);
      const float dist = __fsqrt_rn(u);
      w = __fdiv_rn(1.0f, __fadd_rn(dist, a.eps));
    }
    if (lane < 2 * M) S.lab[c][lane] = __fmul_rn(w, l);
    if (lane == 0) { S.ckey[c] = id < 0 ? 0ull : fin_key(sx, id); S.w[c] = w; }
  }
  __syncthreads();
  // rank by counting (keys are distinct because indices are): warp c ranks candidate c, lane j compares candidate j0 + j;
  // the candidate's weighted labels move to its rank's row
#pragma unroll 1
  for (int c = warp; c < kc; c += nwarps) {
    const unsigned long long me = S.ckey[c];
    int rank = 0;
#pragma unroll 1
    for (int j0 = 0; j0 < kc; j0 += 32) {
      const int j = j0 + lane;
      const unsigned long long other = j < kc ? S.ckey[j] : 0ull;
      rank += __popc(__ballot_sync(0xffffffffu, j < kc && ((other > me) || (other == me && j < c))));
    }
    if (rank < k) {
      if (lane < 2 * M) S.prod[rank][lane] = S.lab[c][lane];
      if (lane == 0) {
        S.wr[rank] = S.w[c];
        if (cp->nn_idx) cp->nn_idx[(size_t)r * k + rank] = me ? (int32_t)(0xffffffffu - (uint32_t)me) : -1;
        if (cp->nn_sim) cp->nn_sim[(size_t)r * k + rank] = me ? rb_o2f((uint32_t)(me >> 32)) : -INFINITY;
      }
    }
  }
  __syncthreads();
  if (warp == 0) {
    // ---- aggregate: lane m < M -> quality, M <= lane < 2M -> output length; the sums are sequential (canonical order) ----
    if (lane < 2 * M) {
      float num = 0.0f, den = 0.0f;
#pragma unroll 4
      for (int j = 0; j < k; ++j) {
        num = __fadd_rn(num, S.prod[j][lane]);
        den = __fadd_rn(den, S.wr[j]);
      }
      const float pred = __fdiv_rn(num, den);
      float* const out_pq = cp->pred_q;
      float* const out_pl = cp->pred_l;
      if (lane < M) {
        S.Q[lane] = pred;
        a.pred_q[(size_t)r * M + lane] = pred;
        if (out_pq) out_pq[(size_t)r * M + lane] = pred;
      } else {
        S.L[lane - M] = pred;
        a.pred_l[(size_t)r * M + lane - M] = pred;
        if (out_pl) out_pl[(size_t)r * M + lane - M] = pred;
      }
    }
    if (a.with_terms) {
      // ---- per-(request, tier) terms: lane = tier ----
      const uint32_t present = __ballot_sync(0xffffffffu, c_present != 0);   // lanes 0..M-1 hold the tiers' flags
      __syncwarp();
      const int m = lane < M ? lane : 0;
      const float L = S.L[m];
      const float C = __fadd_rn(__fmul_rn(c_ell, c_pin), __fmul_rn(L, c_pout));
      float kmax;
      const float A = tier_term_A_warp(lane, present, C, L, S.Q[m], cp->w_qual, cp->w_cost, has_budget, c_budget, &kmax);
      if (lane < M) {
        a.termA[(size_t)r * M + lane] = A;
        a.termP[(size_t)r * M + lane] = __fmul_rn(c_pre, c_ell);
        if (lane == 0) a.key[r] = kmax;
      }
    }
  }
}

}  // namespace
}  // namespace rb
