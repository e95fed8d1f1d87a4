// estimate.cu -- the estimate stage around the tensor-core scan: query staging (a0), the exact fp32-storage
// scan (a1, small banks), and the per-query finishing kernel: cross-CTA top-k merge (a2), exact re-rank +
// distance-weighted aggregate (a3) and the per-(request, tier) score terms (a4).
// Citations: P:L115 (§4.2 "Model estimator"); readings 1-8 and "Canonical arithmetic".
#include "rb_internal.cuh"

namespace rb {
namespace {


// Total order of candidates: similarity descending, bank index ascending (reading 3), as one 64-bit key whose
// unsigned order is that order (larger key = better).  Key 0 is below every real candidate.
__device__ __forceinline__ uint32_t f32_ordered(float f) {
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float f32_unordered(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
__device__ __forceinline__ unsigned long long make_key(float sim, int32_t idx) {
  return ((unsigned long long)f32_ordered(sim) << 32) | (unsigned long long)(0xffffffffu - (uint32_t)idx);
}

// ---- a0 ---------------------------------------------------------------------------------------------
__global__ void stage_queries_kernel(const __grid_constant__ CallParams cpv, __nv_bfloat16* __restrict__ qs, int B, int Bpad,
                                     int d, int group, uint32_t* __restrict__ gthr, int n_gthr, InstTable t,
                                     float* __restrict__ dq, int32_t* __restrict__ bq) {
  const CallParams* __restrict__ cp = &cpv;   // the per-call parameters travel as a kernel argument (constant bank)
  launch_dependents();
  if (blockIdx.x == 0) {
    // a8 folded in: rb_advance_state calls since the last decision (reading 22; same arithmetic as advance_kernel):
    //   tpot = dec*(1 + slope*(float)b); q = dt/tpot; done = (float)b*q; d = max(d - done, 0); if d == 0: b = 0   (b > 0 only)
    const int n_adv = cp->n_adv;
    if (n_adv > 0) {
      for (int i = threadIdx.x; i < t.I; i += blockDim.x) {
        float dd = dq[i];
        int b = bq[i];
        const float dec = t.dec_i[i], slope = t.slope_i[i];
        for (int a = 0; a < n_adv && b > 0; ++a) {
          const float tpot = __fmul_rn(dec, __fadd_rn(1.0f, __fmul_rn(slope, (float)b)));
          const float done = __fmul_rn((float)b, __fdiv_rn(cp->adv_ms[a], tpot));
          dd = fmaxf(__fsub_rn(dd, done), 0.0f);
          if (dd == 0.0f) b = 0;
        }
        dq[i] = dd;
        bq[i] = b;
      }
    }
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_gthr; i += gridDim.x * blockDim.x) gthr[i] = 0u;
  const float* __restrict__ q = cp->query;
  const size_t n = (size_t)Bpad * d;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t row = i / d, c = i - row * d;
    const size_t r = row % group;   // replicas of query r at rows r, group + r, ...
    qs[i] = (r < (size_t)B) ? __float2bfloat16_rn(q[r * d + c]) : __float2bfloat16_rn(0.0f);
  }
}
__global__ void convert_bf16_kernel(const float* __restrict__ in, __nv_bfloat16* __restrict__ out, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = __float2bfloat16_rn(in[i]);
}

// ---- a1, fp32 storage -----------------------------------------------------------------------------------
// s[r,n] = fl32( sum_c (double)x[r,c] * (double)e[n,c] ) in index order: the product of two fp32 values is
// exact in fp64, so one fp64 FMA per term is exactly "multiply, then add with one rounding".
constexpr int kF32Rows = 128;   // bank rows per block, one per thread
constexpr int kF32Q = 8;        // queries per register group
constexpr int kF32Chunk = 64;   // columns staged per step
__global__ void __launch_bounds__(kF32Rows)
scan_f32_kernel(const float* __restrict__ bank, const __grid_constant__ CallParams cpv, int r0, int64_t N, int d, int nq,
                float* __restrict__ sims) {
  __shared__ float xs[kF32Q][kF32Chunk];
  const CallParams* __restrict__ cp = &cpv;
  const float* __restrict__ q = cp->query + (size_t)r0 * d;
  const int64_t n = (int64_t)blockIdx.x * kF32Rows + threadIdx.x;
  const float* row = bank + (n < N ? n : N - 1) * (int64_t)d;
  for (int q0 = 0; q0 < nq; q0 += kF32Q) {
    double acc[kF32Q];
#pragma unroll
    for (int j = 0; j < kF32Q; ++j) acc[j] = 0.0;
    for (int c0 = 0; c0 < d; c0 += kF32Chunk) {
      __syncthreads();
      for (int t = threadIdx.x; t < kF32Q * kF32Chunk; t += kF32Rows) {
        const int j = t / kF32Chunk, c = t % kF32Chunk;
        xs[j][c] = (q0 + j < nq && c0 + c < d) ? q[(size_t)(q0 + j) * d + c0 + c] : 0.0f;
      }
      __syncthreads();
      const int cn = min(kF32Chunk, d - c0);
      for (int c = 0; c < cn; c += 4) {
        const float4 e = *reinterpret_cast<const float4*>(row + c0 + c);
#pragma unroll
        for (int j = 0; j < kF32Q; ++j) {
          acc[j] = fma((double)xs[j][c + 0], (double)e.x, acc[j]);
          acc[j] = fma((double)xs[j][c + 1], (double)e.y, acc[j]);
          acc[j] = fma((double)xs[j][c + 2], (double)e.z, acc[j]);
          acc[j] = fma((double)xs[j][c + 3], (double)e.w, acc[j]);
        }
      }
    }
    if (n < N) {
#pragma unroll
      for (int j = 0; j < kF32Q; ++j)
        if (q0 + j < nq) sims[(size_t)(q0 + j) * N + n] = (float)acc[j];
    }
  }
}

// One block per query: kc rounds, each takes the best row strictly after the previous pick in the total order.
__global__ void __launch_bounds__(256)
select_f32_kernel(const float* __restrict__ sims, int64_t N, int kc, float* __restrict__ cand_sim, int32_t* __restrict__ cand_idx) {
  __shared__ unsigned long long wbest[8];
  __shared__ unsigned long long prev_s;
  const float* s = sims + (size_t)blockIdx.x * N;
  unsigned long long prev = ~0ull;
  for (int j = 0; j < kc; ++j) {
    unsigned long long best = 0;
    for (int64_t n = threadIdx.x; n < N; n += blockDim.x) {
      const float v = s[n];
      if (v == v) {   // NaN never selected
        const unsigned long long key = make_key(v, (int32_t)n);
        if (key < prev && key > best) best = key;
      }
    }
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long other = __shfl_xor_sync(0xffffffffu, best, o);
      best = other > best ? other : best;
    }
    if ((threadIdx.x & 31) == 0) wbest[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
      unsigned long long b = 0;
      for (int w = 0; w < 8; ++w) b = wbest[w] > b ? wbest[w] : b;
      prev_s = b;
      const size_t o = (size_t)blockIdx.x * kc + j;
      if (b == 0) {
        cand_sim[o] = -INFINITY;
        cand_idx[o] = -1;
      } else {
        cand_sim[o] = f32_unordered((uint32_t)(b >> 32));
        cand_idx[o] = (int32_t)(0xffffffffu - (uint32_t)b);
      }
    }
    __syncthreads();
    prev = prev_s;
    if (prev == 0) prev = 1;   // exhausted: later rounds find nothing
  }
}

// ---- a2 + a3 + a4 ---------------------------------------------------------------------------------------
// One CTA per query.  The kernel is bound by the length of its once-executed instruction stream (a cold kernel
// fetches every instruction it executes, and an SM's instruction cache holds 32 KB), so every phase is a short rolled
// loop and the rare cases live in functions that are not inlined.
//  load    the query's partial lists (sorted by key, descending) become 64-bit keys in shared memory.
//  bound   every 8 lanes form a group; the kc-th largest group maximum is reached by kc distinct entries, so every
//          member of the kc best reaches it too (admission bound).
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
constexpr int kFinThreadsMax = 1024;
constexpr int kFinWarpsMax = kFinThreadsMax / 32;
constexpr int kMaxFlag = 16;                      // flagged lists per query <= kc / kcap
constexpr int kSurvMax = 256;                     // survivors of the admission bound that are ranked by counting
constexpr int kGroupsMax = kFinThreadsMax / 8;    // admission groups: 8 lanes each
constexpr int kRescanKeep = 64;                   // entries every warp keeps of a slab it searches again (>= kMaxK)

// s = fl32( sum_c (double)x[c]*(double)e[c] ) of two bf16 rows, the 32 lanes' fp64 partials added by shuffles.
__device__ __forceinline__ float exact_sim_bf16(const uint4* __restrict__ qrow, const uint4* __restrict__ brow, int nvec,
                                                int lane) {
  double acc = 0.0;
#pragma unroll 2
  for (int vidx = lane; vidx < nvec; vidx += 32) {
    const uint4 xb = qrow[vidx], eb = brow[vidx];
    const __nv_bfloat162* xp = reinterpret_cast<const __nv_bfloat162*>(&xb);
    const __nv_bfloat162* ep = reinterpret_cast<const __nv_bfloat162*>(&eb);
#pragma unroll
    for (int h = 0; h < 4; ++h) {
      const float2 xf = __bfloat1622float2(xp[h]), ef = __bfloat1622float2(ep[h]);
      acc = fma((double)xf.x, (double)ef.x, acc);
      acc = fma((double)xf.y, (double)ef.y, acc);
    }
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  return (float)acc;
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
// searched again with exact similarities; s_cand becomes the kc best of those slabs' rows and of the candidates that
// came from the other slabs.  s_keys is overwritten ([nwarps][kRescanKeep] + [kc]).  All threads must call; rare path.
__device__ __noinline__ void rescan_slabs(const FinishArgs& a, const uint4* qrow, int nvec, unsigned long long kstar,
                                          unsigned long long* s_keys, unsigned long long* s_cand,
                                          uint32_t (*s_red)[kFinWarpsMax][2], int* s_flag, int* s_nflag) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nwarps = blockDim.x >> 5;
  const int kc = a.kc, kcap = a.kcap;
  if (tid == 0) *s_nflag = 0;
  __syncthreads();
  for (int l = tid; l < a.nlists; l += blockDim.x) {
    const unsigned long long last = s_keys[(size_t)l * kcap + kcap - 1];
    if (last != 0ull && last >= kstar) {
      const int p = atomicAdd(s_nflag, 1);
      if (p < kMaxFlag) s_flag[p] = l / a.lists_per_cta;
    }
  }
  __syncthreads();
  if (tid == 0) {   // lists -> slabs, each once
    const int nl = min(*s_nflag, kMaxFlag);
    int nc = 0;
    for (int f = 0; f < nl; ++f) {
      const int c = s_flag[f];
      bool seen = false;
      for (int g = 0; g < nc; ++g) seen |= (s_flag[g] == c);
      if (!seen) s_flag[nc++] = c;
    }
    *s_nflag = nc;
  }
  __syncthreads();
  const int nflag = *s_nflag;
  const int nslabs = a.nlists / a.lists_per_cta;
  // every warp keeps the best 64 of the rows it visits: rank l in lane l (la) and rank 32 + l (lb)
  unsigned long long la = 0, lb = 0, thr = 0;
  for (int f = 0; f < nflag; ++f) {
    int64_t row0, row1;
    slab_rows(a, s_flag[f], nslabs, &row0, &row1);
    for (int64_t n = row0 + warp; n < row1; n += nwarps) {
      const float sx = exact_sim_bf16(qrow, reinterpret_cast<const uint4*>(a.bank + (size_t)n * a.d), nvec, lane);
      const unsigned long long x = make_key(sx, (int32_t)n);
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
    const unsigned long long key = s_cand[tid];
    bool from_flagged = false;
    if (key != 0ull) {
      const int64_t n = (int64_t)(0xffffffffu - (uint32_t)key);
      for (int f = 0; f < nflag; ++f) {
        int64_t row0, row1;
        slab_rows(a, s_flag[f], nslabs, &row0, &row1);
        from_flagged |= (n >= row0 && n < row1);
      }
    }
    s_keys[(size_t)nwarps * kRescanKeep + tid] = from_flagged ? 0ull : key;
  }
  __syncthreads();
  block_select_topk(s_keys, nwarps * kRescanKeep + kc, kc, s_red, s_cand);
}

__global__ void __launch_bounds__(kFinThreadsMax)
finish_kernel(FinishArgs a, InstTable t, const __grid_constant__ CallParams cpv) {
  const CallParams* __restrict__ cp = &cpv;   // per-call parameters: a kernel argument (constant bank), not a device block
  extern __shared__ unsigned long long s_keys[];   // max([nlists][kcap], [nwarps][kRescanKeep] + [kMaxK])
  __shared__ uint32_t s_red[2][kFinWarpsMax][2];
  __shared__ uint32_t s_gmax[kGroupsMax];
  __shared__ unsigned long long s_surv[kSurvMax];
  __shared__ unsigned long long s_cand[kMaxK];
  __shared__ int s_nsurv, s_nflag;
  __shared__ uint32_t s_tau;
  __shared__ int s_flag[kMaxFlag];
  __shared__ float s_sim[kMaxK];
  __shared__ int32_t s_idx[kMaxK];
  __shared__ float s_w[kMaxK];
  __shared__ float s_lab[kMaxK][2 * kMaxM];         // labels of the kc candidates: [quality(M) | outlen(M)]
  __shared__ int s_pos[kMaxK];                      // candidate at each final rank
  __shared__ float sQ[kMaxM], sL[kMaxM];
  const int r = blockIdx.x;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nthreads = blockDim.x, nwarps = blockDim.x >> 5;
  // coefficients of the score terms: requested now, consumed at the very end (their latency hides behind the merge)
  float c_pin = 0.0f, c_pout = 0.0f, c_pre = 0.0f, c_ell = 0.0f, c_budget = 0.0f;
  bool has_budget = false;
  int c_present = 0;
  if (a.with_terms && tid < a.M) {
    c_pin = t.price_in[tid];
    c_pout = t.price_out[tid];
    c_pre = t.pre[tid];
    c_present = t.present[tid];
    c_ell = (float)cp->plen[r];
    has_budget = cp->budget != nullptr;
    if (has_budget) c_budget = cp->budget[r];
  }
  const int kc = a.kc, k = a.k, kcap = a.kcap, M = a.M;
  const uint4* qrow = reinterpret_cast<const uint4*>(a.qs + (size_t)r * a.d);
  const int nvec = a.d / 8;   // d % 8 == 0
  const int total = a.nlists * kcap;
  if (tid == 0) s_nsurv = 0;
  launch_dependents();
  grid_dependency_wait();   // the partial lists come from the preceding kernel

  // ---- load: lists -> keys in shared memory; every thread remembers the best similarity it has seen ----
  uint32_t tmax = 0u;
  if (kcap & 3) {   // one already-merged list per query, entry by entry ([nlists][Bpad][kcap] arrays)
    for (int e = tid; e < total; e += nthreads) {
      const int c = e / kcap, j = e - c * kcap;
      const size_t off = ((size_t)c * a.Bpad + r) * kcap + j;
      const int32_t id = a.part_idx[off];
      const unsigned long long key = (id >= 0 && (int64_t)id < a.N) ? make_key(a.part_sim[off], id) : 0ull;
      s_keys[e] = key;
      tmax = max(tmax, (uint32_t)(key >> 32));
    }
  } else {
    // a list's kcap entries are contiguous (kcap is a multiple of 4): one quad = 4 similarities + 4 indices per step
    const int q4 = kcap >> 2, nquads = a.nlists * q4;
#pragma unroll 1
    for (int e = tid; e < nquads; e += nthreads) {
      uint4 ua, ub;
      if (a.records) {   // record e of this query: [4 similarities | 4 indices], contiguous over e (one run per query)
        const uint4* rec = reinterpret_cast<const uint4*>(a.part_sim) + ((size_t)r * nquads + e) * 2;
        ua = __ldcg(rec);
        ub = __ldcg(rec + 1);
      } else {
        const int c = e / q4, j4 = e - c * q4;
        const size_t off = ((size_t)c * a.Bpad + r) * kcap + 4 * j4;
        ua = __ldcg(reinterpret_cast<const uint4*>(a.part_sim + off));
        ub = __ldcg(reinterpret_cast<const uint4*>(a.part_idx + off));
      }
      const uint32_t sx[4] = {ua.x, ua.y, ua.z, ua.w};
      const uint32_t ix[4] = {ub.x, ub.y, ub.z, ub.w};
#pragma unroll
      for (int h = 0; h < 4; ++h) {
        const int32_t id = (int32_t)ix[h];
        const unsigned long long key = (id >= 0 && (int64_t)id < a.N) ? make_key(__uint_as_float(sx[h]), id) : 0ull;
        s_keys[4 * e + h] = key;
        tmax = max(tmax, (uint32_t)(key >> 32));
      }
    }
  }
  // ---- bound: kc-th largest of the 8-lane group maxima ----
  tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
  tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
  tmax = max(tmax, __shfl_xor_sync(0xffffffffu, tmax, 4));
  const int ngroups = nthreads >> 3;
  if ((lane & 7) == 0) s_gmax[tid >> 3] = tmax;
  if (tid == 0) s_tau = 0u;
  __syncthreads();
  if (tid < ngroups && ngroups >= kc) {
    const uint32_t mine = s_gmax[tid];
    int rank = 0;
#pragma unroll 4
    for (int g = 0; g < ngroups; ++g) {
      const uint32_t o = s_gmax[g];
      rank += (o > mine) || (o == mine && g < tid);
    }
    if (rank == kc - 1) s_tau = mine;   // ranks are distinct: exactly one writer
  }
  __syncthreads();
  // ---- select: survivors of the bound, compacted ----
  const uint32_t tau = s_tau;
  // (every thread revisits the entries it wrote itself: quads tid, tid + nthreads, ...)
  if (kcap & 3) {
    for (int e = tid; e < total; e += nthreads) {
      const unsigned long long key = s_keys[e];
      if (key != 0ull && (uint32_t)(key >> 32) >= tau) {
        const int p = atomicAdd(&s_nsurv, 1);
        if (p < kSurvMax) s_surv[p] = key;
      }
    }
  } else {
    const int nquads = total >> 2;
#pragma unroll 1
    for (int e = tid; e < nquads; e += nthreads) {
#pragma unroll 1
      for (int h = 0; h < 4; ++h) {   // a list is sorted: stop at the first entry below the bound
        const unsigned long long key = s_keys[4 * e + h];
        if (key == 0ull || (uint32_t)(key >> 32) < tau) break;
        const int p = atomicAdd(&s_nsurv, 1);
        if (p < kSurvMax) s_surv[p] = key;
      }
    }
  }
  __syncthreads();
  const int nsurv = s_nsurv;
  if (nsurv <= kSurvMax) {
    // rank by counting: thread c ranks survivor c
    if (tid < kc) s_cand[tid] = 0ull;
    __syncthreads();
    if (tid < nsurv) {
      const unsigned long long mine = s_surv[tid];
      int rank = 0;
#pragma unroll 4
      for (int j = 0; j < nsurv; ++j) rank += s_surv[j] > mine;
      if (rank < kc) s_cand[rank] = mine;
    }
    __syncthreads();
  } else {
    block_select_topk(s_keys, total, kc, s_red, s_cand);
  }
  // ---- rescan of slabs whose list may hide members ----
  if (a.rescan) {
    const unsigned long long kstar = s_cand[kc - 1];
    bool flagged = false;
    for (int l = tid; l < a.nlists; l += nthreads) {
      const unsigned long long last = s_keys[(size_t)l * kcap + kcap - 1];
      flagged |= (last != 0ull && last >= kstar);
    }
    if (__syncthreads_or(flagged)) rescan_slabs(a, qrow, nvec, kstar, s_keys, s_cand, s_red, s_flag, &s_nflag);
  }

  // ---- exact re-rank: warp c recomputes candidate c (and gathers its labels meanwhile) ----
  float* const out_pq = cp->pred_q;
  float* const out_pl = cp->pred_l;
  int32_t* const out_nn_idx = cp->nn_idx;
  float* const out_nn_sim = cp->nn_sim;
#pragma unroll 1
  for (int c = warp; c < kc; c += nwarps) {
    const unsigned long long key = s_cand[c];
    const int32_t id = key ? (int32_t)(0xffffffffu - (uint32_t)key) : -1;
    float sx = key ? f32_unordered((uint32_t)(key >> 32)) : -INFINITY;
    float lv = 0.0f;   // the candidate's labels are requested first: independent of the bank row's loads
    if (id >= 0 && lane < 2 * M) lv = (lane < M) ? a.bank_quality[(size_t)id * M + lane] : a.bank_outlen[(size_t)id * M + lane - M];
    if (id >= 0 && a.rerank) sx = exact_sim_bf16(qrow, reinterpret_cast<const uint4*>(a.bank + (size_t)id * a.d), nvec, lane);
    if (lane == 0) { s_sim[c] = sx; s_idx[c] = id; }
    if (lane < 2 * M) s_lab[c][lane] = lv;
  }
  __syncthreads();
  // rank by counting (keys are distinct because indices are): warp c ranks candidate c, lane j compares candidate j;
  // lane 0 then computes the weight of the rank-th neighbour (the warps' square roots and divisions overlap)
#pragma unroll 1
  for (int c = warp; c < kc; c += nwarps) {
    const int32_t id = s_idx[c];
    const float sc = s_sim[c];
    const unsigned long long me = (id < 0) ? 0ull : make_key(sc, id);
    int rank = 0;
    for (int j0 = 0; j0 < kc; j0 += 32) {
      const int j = j0 + lane;
      bool ahead = false;
      if (j < kc) {
        const int32_t oj = s_idx[j];
        const unsigned long long other = (oj < 0) ? 0ull : make_key(s_sim[j], oj);
        ahead = (other > me) || (other == me && j < c);
      }
      rank += __popc(__ballot_sync(0xffffffffu, ahead));
    }
    if (rank < k) {
      if (lane == 0) {
        s_pos[rank] = c;
        float w = 1.0f;
        if (id < 0) {
          w = 0.0f;   // fewer than k rows reachable (cannot happen for k <= N); adds +0 to both sums
        } else if (a.weight_mode == 0) {
          const float tt = __fmul_rn(2.0f, sc);
          float u = __fsub_rn(2.0f, tt);
          u = fmaxf(u, 0.0f);
          const float dist = __fsqrt_rn(u);
          w = __fdiv_rn(1.0f, __fadd_rn(dist, a.eps));
        }
        s_w[rank] = w;
        if (out_nn_idx) out_nn_idx[(size_t)r * k + rank] = id;
        if (out_nn_sim) out_nn_sim[(size_t)r * k + rank] = sc;
      }
    }
  }
  __syncthreads();
  if (warp != 0) return;
  // ---- aggregate: lane m < M -> quality, M <= lane < 2M -> output length ----
  if (lane < 2 * M) {
    float num = 0.0f, den = 0.0f;
#pragma unroll 4   // four neighbours' loads in flight; the two sums stay sequential (canonical order)
    for (int j = 0; j < k; ++j) {
      const float w = s_w[j];
      const float p = __fmul_rn(w, s_lab[s_pos[j]][lane]);
      num = __fadd_rn(num, p);
      den = __fadd_rn(den, w);
    }
    const float pred = __fdiv_rn(num, den);
    if (lane < M) {
      sQ[lane] = pred;
      a.pred_q[(size_t)r * M + lane] = pred;
      if (out_pq) out_pq[(size_t)r * M + lane] = pred;
    } else {
      sL[lane - M] = pred;
      a.pred_l[(size_t)r * M + lane - M] = pred;
      if (out_pl) out_pl[(size_t)r * M + lane - M] = pred;
    }
  }
  if (!a.with_terms) return;
  // ---- per-(request, tier) terms: lane = tier ----
  const uint32_t present = __ballot_sync(0xffffffffu, c_present != 0);   // lanes 0..M-1 hold the tiers' flags
  __syncwarp();
  {
    const int m = lane < M ? lane : 0;
    const float L = sL[m];
    const float C = __fadd_rn(__fmul_rn(c_ell, c_pin), __fmul_rn(L, c_pout));
    float kmax;
    const float A = tier_term_A_warp(lane, present, C, L, sQ[m], cp->w_qual, cp->w_cost, has_budget, c_budget, &kmax);
    if (lane < M) {
      a.termA[(size_t)r * M + lane] = A;
      a.termP[(size_t)r * M + lane] = __fmul_rn(c_pre, c_ell);
      if (lane == 0) a.key[r] = kmax;
    }
  }
}

}  // namespace

cudaError_t launch_convert_bf16(const float* in, __nv_bfloat16* out, size_t n, cudaStream_t s) {
  size_t blocks = (n + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  convert_bf16_kernel<<<(int)blocks, 256, 0, s>>>(in, out, n);
  return cudaGetLastError();
}

cudaError_t launch_stage_queries(const CallParams& cp, __nv_bfloat16* qs, int B, int Bpad, int d, int rep, uint32_t* gthr,
                                 int n_gthr, InstTable t, float* dq, int32_t* bq, cudaStream_t s) {
  const size_t n = (size_t)Bpad * d;
  int blocks = (int)((n + 255) / 256);
  if (blocks > 148 * 8) blocks = 148 * 8;
  stage_queries_kernel<<<blocks, 256, 0, s>>>(cp, qs, B, Bpad, d, rep > 1 ? kTileM / rep : Bpad, gthr, n_gthr, t, dq, bq);
  return cudaGetLastError();
}

cudaError_t launch_scan_f32(const float* bank, const CallParams& cp, int r0, int64_t N, int d, int nq, float* sims,
                            cudaStream_t s) {
  const int blocks = (int)((N + kF32Rows - 1) / kF32Rows);
  scan_f32_kernel<<<blocks, kF32Rows, 0, s>>>(bank, cp, r0, N, d, nq, sims);
  return cudaGetLastError();
}

cudaError_t launch_select_f32(const float* sims, int64_t N, int nq, int kc, float* cand_sim, int32_t* cand_idx,
                              cudaStream_t s) {
  select_f32_kernel<<<nq, 256, 0, s>>>(sims, N, kc, cand_sim, cand_idx);
  return cudaGetLastError();
}

// Position and count of the arguments of this file's kernels that carry the per-call parameters (graph replays update
// that one argument): returns the index of the CallParams argument, or -1 if func is not one of them.
int estimate_cp_arg(const void* func, int* nargs) {
  if (func == (const void*)stage_queries_kernel) { *nargs = 11; return 0; }
  if (func == (const void*)scan_f32_kernel) { *nargs = 7; return 1; }
  if (func == (const void*)finish_kernel) { *nargs = 3; return 2; }
  return -1;
}

size_t finish_smem_bytes(int nlists, int kcap) {
  // keys of all lists; the rescan reuses the space for the warps' own lists and the other slabs' candidates
  const size_t n1 = (size_t)nlists * kcap * 8;
  const size_t n2 = (size_t)(kFinWarpsMax * kRescanKeep + kMaxK) * 8;
  return n1 > n2 ? n1 : n2;
}

cudaError_t finish_prepare(size_t max_smem) {
  return cudaFuncSetAttribute(finish_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem);
}

cudaError_t launch_finish(const FinishArgs& a, InstTable t, const CallParams& cp, int B, cudaStream_t s) {
  // one thread per quad of list entries where that fits; at least 16 warps (one per candidate of the re-rank)
  const int nquads = a.nlists * ((a.kcap + 3) / 4);
  const int threads = nquads <= 512 ? 512 : (nquads >= 1024 ? 1024 : (nquads + 31) / 32 * 32);
  const cudaError_t e = launch_chained(finish_kernel, dim3(B), dim3(threads), finish_smem_bytes(a.nlists, a.kcap), s, a, t, cp);
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rb
