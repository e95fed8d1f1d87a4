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
// One CTA per query.
//  merge   the nlists partial lists (each sorted by key, descending) are copied to shared memory as 64-bit
//          keys; thread c owns list c and exposes its head; kc rounds of a block-wide maximum (REDUX on the
//          high and low words, one barrier per round) pop the kc best in order.
//  rescan  the scan may keep fewer entries per (CTA, query) than kc (short lists make its warm-up cheap).  A list
//          whose every entry was popped may hide further members of the top kc; the bank rows of such a slab
//          (rare: several of a query's kc best in one of ~148 slabs) are searched again here, exactly, and the
//          merge is redone over the untouched lists' candidates and the slab's own best kc.
//  re-rank (bf16 storage): the kc candidates' similarities are recomputed from the stored bf16 rows with fp64
//          accumulation (products of bf16 values are exact), rounded once to fp32, re-ordered by
//          (s desc, n asc); the best k are the neighbours.
//  aggregate:
//          t = 2*s; u = 2 - t; u = max(u,0); dist = sqrt(u); w = 1/(dist + eps)      (uniform mode: w = 1)
//          num_m = sum_j w_j*label[n_j,m] (j ascending, multiply then add); den = sum_j w_j; pred = num/den
//  terms   (with_terms; Eq. 2, Eq. 1):
//          c1 = (float)l*pin; c2 = L*pout; C = c1 + c2; Cmax over tiers that have an instance;
//          ct = Cmax > 0 ? 1 - C/Cmax : 0; A = wq*Q + wc*ct; P = pre*(float)l; key = max_m L
constexpr int kFinThreadsMax = 1024;              // 512 threads, or 1024 when there are more than 512 lists
constexpr int kFinWarpsMax = kFinThreadsMax / 32;
constexpr int kMaxFlag = 16;                      // flagged lists per query <= kc / kcap
constexpr int kMerge2Stride = 64;                 // second merge: nwarps + 1 lists of up to kMaxK keys

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

// Warp-level k-way merge: lane l owns the sorted list keys[(first + l)*stride ..] (l < nl <= 32) and the warp
// pops the kc largest keys, in order, into out_key / out_src (the owning list's index).  No block barrier.
// bound_hi: similarity (ordered bits) that every member of the query's kc best reaches (0 = none known): the warp stops
// popping below it and pads the rest of its output with empty entries.
// Returns the number of entries popped (warp-uniform).
__device__ __forceinline__ int warp_kway_merge(const unsigned long long* keys, int first, int nl, int stride, int len,
                                               int kc, unsigned long long* out_key, int* out_src, uint32_t bound_hi) {
  const int lane = threadIdx.x & 31;
  const unsigned long long* mine = keys + (size_t)(first + lane) * stride;
  int pos = 0, npop = 0;
  unsigned long long hk = (lane < nl) ? mine[0] : 0ull;
  for (int j = 0; j < kc; ++j) {
    const uint32_t hi = (uint32_t)(hk >> 32), lo = (uint32_t)hk;
    const uint32_t ghi = __reduce_max_sync(0xffffffffu, hi);
    if (ghi < bound_hi) {   // warp-uniform: nothing left here can be among the kc best
      for (int jj = j + lane; jj < kc; jj += 32) { out_key[jj] = 0ull; out_src[jj] = -1; }
      break;
    }
    npop += ghi != 0u;
    const uint32_t glo = __reduce_max_sync(0xffffffffu, hi == ghi ? lo : 0u);
    const unsigned long long win = ((unsigned long long)ghi << 32) | glo;
    if (win != 0ull && hk == win) {   // keys are distinct: exactly one owner
      out_key[j] = win;
      out_src[j] = first + lane;
      ++pos;
      hk = pos < len ? mine[pos] : 0ull;
    }
    if (win == 0ull && lane == 0) { out_key[j] = 0ull; out_src[j] = -1; }
  }
  return npop;
}

// Block-wide k-way merge: thread c < nl owns the sorted list keys[c*stride .. c*stride+len); pops the kc largest
// keys into out_key[0..kc) (0 = exhausted) and the list each came from into out_src.  Returns how many entries
// of the caller's own list were popped.  All threads of the block must call.
__device__ int kway_merge(const unsigned long long* keys, int nl, int stride, int len, int kc,
                          uint32_t (*s_red)[kFinWarpsMax][2], unsigned long long* out_key, int* out_src) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, kFinWarps = blockDim.x >> 5;
  int pos = 0;
  unsigned long long hk = (tid < nl) ? keys[(size_t)tid * stride] : 0ull;
  for (int j = 0; j < kc; ++j) {
    const uint32_t hi = (uint32_t)(hk >> 32), lo = (uint32_t)hk;
    const uint32_t whi = __reduce_max_sync(0xffffffffu, hi);
    const uint32_t wlo = __reduce_max_sync(0xffffffffu, hi == whi ? lo : 0u);
    if (lane == 0) { s_red[j & 1][warp][0] = whi; s_red[j & 1][warp][1] = wlo; }
    __syncthreads();
    const uint32_t xhi = lane < kFinWarps ? s_red[j & 1][lane][0] : 0u;
    const uint32_t xlo = lane < kFinWarps ? s_red[j & 1][lane][1] : 0u;
    const uint32_t ghi = __reduce_max_sync(0xffffffffu, xhi);
    const uint32_t glo = __reduce_max_sync(0xffffffffu, xhi == ghi ? xlo : 0u);
    const unsigned long long win = ((unsigned long long)ghi << 32) | glo;
    if (win != 0ull && hk == win) {   // keys are distinct: exactly one owner
      out_key[j] = win;
      out_src[j] = tid;
      ++pos;
      hk = pos < len ? keys[(size_t)tid * stride + pos] : 0ull;
    }
    if (win == 0ull && tid == 0) { out_key[j] = 0ull; out_src[j] = -1; }
  }
  __syncthreads();
  return pos;
}

__global__ void __launch_bounds__(kFinThreadsMax)
finish_kernel(FinishArgs a, InstTable t, const __grid_constant__ CallParams cpv) {
  const CallParams* __restrict__ cp = &cpv;   // per-call parameters: a kernel argument (constant bank), not a device block
  extern __shared__ unsigned long long s_keys[];   // max([nlists][kcap], [nwarps + 1][kMerge2Stride])
  __shared__ uint32_t s_red[2][kFinWarpsMax][2];
  __shared__ unsigned long long s_cand[kMaxK];
  __shared__ int s_src[kMaxK];
  __shared__ int s_nflag;
  __shared__ uint32_t s_wbest[kFinWarpsMax];
  __shared__ int s_maxcnt;
  __shared__ int s_wcnt[kFinWarpsMax];                // entries each warp popped at the first level
  __shared__ unsigned long long s_skey[64];           // first-level survivors, compacted (second level by counting)
  __shared__ int s_ssrc[64];
  __shared__ int s_flag[kMaxFlag];
  __shared__ float s_sim[kMaxK];
  __shared__ int32_t s_idx[kMaxK];
  __shared__ float o_sim[kMaxK];
  __shared__ int32_t o_idx[kMaxK];
  __shared__ float s_w[kMaxK];
  __shared__ int o_pos[kMaxK];
  __shared__ float s_lab[kMaxK][2 * kMaxM];         // labels of the kc candidates: [quality(M) | outlen(M)]
  __shared__ float sQ[kMaxM], sL[kMaxM];
  const int r = blockIdx.x;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int kFinThreads = blockDim.x, nwarps = blockDim.x >> 5;
  // coefficients of the score terms: requested now, consumed at the very end (their latency hides behind the merge)
  float c_pin = 0.0f, c_pout = 0.0f, c_pre = 0.0f, c_ell = 0.0f, c_budget = 0.0f;
  bool has_budget = false;
  if (a.with_terms && tid < a.M) {
    c_pin = t.price_in[tid];
    c_pout = t.price_out[tid];
    c_pre = t.pre[tid];
    c_ell = (float)cp->plen[r];
    has_budget = cp->budget != nullptr;
    if (has_budget) c_budget = cp->budget[r];
  }
  const int c_present = (a.with_terms && tid < a.M) ? t.present[tid] : 0;
  // caller-side output pointers and weights: read once, up front (every later use would be an L2 round trip)
  float* const out_pq = cp->pred_q;
  float* const out_pl = cp->pred_l;
  int32_t* const out_nn_idx = cp->nn_idx;
  float* const out_nn_sim = cp->nn_sim;
  const float c_wq = cp->w_qual, c_wc = cp->w_cost;
  const int kc = a.kc, k = a.k, kcap = a.kcap, M = a.M;
  const uint4* qrow = reinterpret_cast<const uint4*>(a.qs + (size_t)r * a.d);
  const int nvec = a.d / 8;   // d % 8 == 0

  // ---- merge ----
  const int total = a.nlists * kcap;
  launch_dependents();
  grid_dependency_wait();   // the partial lists come from the preceding kernel
  if (tid == 0) s_nflag = 0;
  if (kcap & 3) {   // fp32-storage path: one already-merged list of kc entries per query
    for (int e = tid; e < total; e += kFinThreads) {
      const int c = e / kcap, j = e - c * kcap;
      const size_t off = ((size_t)c * a.Bpad + r) * kcap + j;
      const int32_t id = a.part_idx[off];
      s_keys[e] = (id >= 0 && (int64_t)id < a.N) ? make_key(a.part_sim[off], id) : 0ull;
    }
  } else {
    // a list's kcap entries are contiguous (kcap is a multiple of 4): one 16-byte load of similarities and one of
    // indices per (list, quad); two quads in flight per thread
    const int q4 = kcap >> 2, nquads = a.nlists * q4;
    for (int e0 = tid; e0 < nquads; e0 += 2 * kFinThreads) {
      float4 sv[2];
      int4 iv[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int e = e0 + u * kFinThreads;
        if (e < nquads) {
          if (a.records) {   // record e of this query: [4 similarities | 4 indices], contiguous over e
            // (a list-major layout of the same records was tried: the 4 KB stride between a query's records costs the
            // finishing CTA ~3000 cycles more than this contiguous run)
            const uint4* rec = reinterpret_cast<const uint4*>(a.part_sim) + ((size_t)r * nquads + e) * 2;
            const uint4 ua = __ldcg(rec), ub = __ldcg(rec + 1);
            sv[u] = make_float4(__uint_as_float(ua.x), __uint_as_float(ua.y), __uint_as_float(ua.z), __uint_as_float(ua.w));
            iv[u] = make_int4((int)ub.x, (int)ub.y, (int)ub.z, (int)ub.w);
          } else {
            const int c = e / q4, j4 = e - c * q4;
            const size_t off = ((size_t)c * a.Bpad + r) * kcap + 4 * j4;
            sv[u] = __ldcg(reinterpret_cast<const float4*>(a.part_sim + off));
            iv[u] = __ldcg(reinterpret_cast<const int4*>(a.part_idx + off));
          }
        }
      }
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int e = e0 + u * kFinThreads;
        if (e < nquads) {
          const float sx[4] = {sv[u].x, sv[u].y, sv[u].z, sv[u].w};
          const int32_t ix[4] = {iv[u].x, iv[u].y, iv[u].z, iv[u].w};
#pragma unroll
          for (int h = 0; h < 4; ++h)
            s_keys[4 * e + h] = (ix[h] >= 0 && (int64_t)ix[h] < a.N) ? make_key(sx[h], ix[h]) : 0ull;
        }
      }
    }
  }
  __syncthreads();
  // two levels, no barrier inside either: every warp pops the kc best of its own share of the lists (lane = list),
  // then warp 0 pops the kc best of the warps' results (lane = warp)
  unsigned long long* w_key = s_keys + total;                         // [nwarps][kMerge2Stride]
  int* w_src = reinterpret_cast<int*>(w_key + (size_t)nwarps * kMerge2Stride);   // [nwarps][kMerge2Stride]
  {
    const int per = (a.nlists + nwarps - 1) / nwarps;                 // <= 32 by the choice of the block size
    const int first = warp * per;
    const int nl = max(0, min(per, a.nlists - first));
    // Admission bound: the kc-th largest of the warps' best similarities is reached by kc distinct candidates, so
    // every member of the kc best reaches it too -- a warp then pops two or three entries instead of kc.
    uint32_t bound = 0u;
    if (nwarps >= kc) {   // block-uniform
      const uint32_t head = lane < nl ? (uint32_t)(s_keys[(size_t)(first + lane) * kcap] >> 32) : 0u;
      const uint32_t wbest = __reduce_max_sync(0xffffffffu, head);
      if (lane == 0) s_wbest[warp] = wbest;
      __syncthreads();
      uint32_t v = lane < nwarps ? s_wbest[lane] : 0u;
#pragma unroll
      for (int size = 2; size <= 32; size <<= 1) {
#pragma unroll
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
          const uint32_t other = __shfl_xor_sync(0xffffffffu, v, stride);
          const bool keep_max = ((lane & stride) == 0) == ((lane & size) == 0);   // descending
          v = (keep_max == (v > other)) ? v : other;
        }
      }
      bound = __shfl_sync(0xffffffffu, v, kc - 1);
    }
    const int npop = warp_kway_merge(s_keys, first, nl, kcap, kcap, kc, w_key + (size_t)warp * kMerge2Stride,
                                     w_src + (size_t)warp * kMerge2Stride, bound);
    if (lane == 0) s_wcnt[warp] = npop;
  }
  __syncthreads();
  if (warp == 0) {
    // out_src of this level is the warp whose list the key came from; its position in that list is the number
    // of keys already taken from it, which recovers the original list index
    const unsigned long long* mine = w_key + (size_t)lane * kMerge2Stride;
    // With the admission bound the warps hand over a few dozen entries in all: rank them by counting (keys are
    // distinct) instead of kc sequential pops.  More than 64 (no bound, or a bank sorted by topic): the pops below.
    const int cnt = lane < nwarps ? s_wcnt[lane] : 0;
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int up = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += up;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    // a list can only have been popped completely if its warp popped at least kcap entries
    const int maxcnt = (int)__reduce_max_sync(0xffffffffu, (uint32_t)cnt);
    if (lane == 0) s_maxcnt = maxcnt;
    if (total <= 64) {
      const int off = incl - cnt;
      for (int q = 0; q < cnt; ++q) {
        s_skey[off + q] = mine[q];
        s_ssrc[off + q] = w_src[(size_t)lane * kMerge2Stride + q];
      }
      __syncwarp();
      const unsigned long long k0 = lane < total ? s_skey[lane] : 0ull, k1 = lane + 32 < total ? s_skey[lane + 32] : 0ull;
      int rk0 = 0, rk1 = 0;
      for (int q = 0; q < total; ++q) {
        const unsigned long long o = s_skey[q];
        rk0 += o > k0;
        rk1 += o > k1;
      }
      if (lane < total && rk0 < kc) { s_cand[rk0] = k0; s_src[rk0] = s_ssrc[lane]; }
      if (lane + 32 < total && rk1 < kc) { s_cand[rk1] = k1; s_src[rk1] = s_ssrc[lane + 32]; }
      for (int j = total + lane; j < kc; j += 32) { s_cand[j] = 0ull; s_src[j] = -1; }
    } else {
    int pos = 0;
    unsigned long long hk = (lane < nwarps) ? mine[0] : 0ull;
    for (int j = 0; j < kc; ++j) {
      const uint32_t hi = (uint32_t)(hk >> 32), lo = (uint32_t)hk;
      const uint32_t ghi = __reduce_max_sync(0xffffffffu, hi);
      const uint32_t glo = __reduce_max_sync(0xffffffffu, hi == ghi ? lo : 0u);
      const unsigned long long win = ((unsigned long long)ghi << 32) | glo;
      if (win != 0ull && hk == win) {
        s_cand[j] = win;
        s_src[j] = w_src[(size_t)lane * kMerge2Stride + pos];
        ++pos;
        hk = pos < kc ? mine[pos] : 0ull;
      }
      if (win == 0ull && lane == 0) { s_cand[j] = 0ull; s_src[j] = -1; }
    }
    }
  }
  __syncthreads();

  // ---- rescan of slabs whose list was popped completely ----
  // (a list of kcap entries all of which are among the kc best may hide further members)
  bool flagged = false;
  if (a.rescan && s_maxcnt >= kcap && tid < kc && s_src[tid] >= 0) {
    int same = 0, earlier = 0;
    for (int j = 0; j < kc; ++j) {
      same += (s_src[j] == s_src[tid]);
      earlier += (j < tid && s_src[j] == s_src[tid]);
    }
    flagged = (same == kcap) && (earlier == 0);
  }
  if (__syncthreads_or(flagged)) {
    if (flagged) {
      const int p = atomicAdd(&s_nflag, 1);
      if (p < kMaxFlag) s_flag[p] = s_src[tid];
    }
    __syncthreads();
    if (tid == 0) {   // lists -> CTAs (slabs), each once
      const int nl = min(s_nflag, kMaxFlag);
      int nc = 0;
      for (int f = 0; f < nl; ++f) {
        const int c = s_flag[f] / a.lists_per_cta;
        bool seen = false;
        for (int g = 0; g < nc; ++g) seen |= (s_flag[g] == c);
        if (!seen) s_flag[nc++] = c;
      }
      s_nflag = nc;
    }
    __syncthreads();
    const int nflag = s_nflag;
    const int nctas = a.nlists / a.lists_per_cta;
    // every warp keeps the best kc of the rows it visits: rank l in lane l (a) and rank 32+l (b)
    unsigned long long la = 0, lb = 0, thr = 0;
    const int64_t units = (a.N + a.slab_unit - 1) / a.slab_unit;
    for (int f = 0; f < nflag; ++f) {
      const int c = s_flag[f];
      const int64_t row0 = units * c / nctas * a.slab_unit;
      int64_t row1 = units * (c + 1) / nctas * a.slab_unit;
      if (row1 > a.N) row1 = a.N;
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
    __syncthreads();   // s_keys is rewritten: lists 0..nwarps-1 = the warps' lists, list nwarps = untouched candidates
    s_keys[(size_t)warp * kMerge2Stride + lane] = la;
    s_keys[(size_t)warp * kMerge2Stride + 32 + lane] = lb;
    if (tid == 0) {
      int o = 0;
      for (int j = 0; j < kc; ++j) {
        bool from_flagged = false;
        for (int f = 0; f < nflag; ++f) from_flagged |= (s_src[j] / a.lists_per_cta == s_flag[f]);
        if (s_cand[j] != 0ull && !from_flagged) s_keys[(size_t)nwarps * kMerge2Stride + o++] = s_cand[j];
      }
      for (; o < kMerge2Stride; ++o) s_keys[(size_t)nwarps * kMerge2Stride + o] = 0ull;
    }
    __syncthreads();
    kway_merge(s_keys, nwarps + 1, kMerge2Stride, kMerge2Stride, kc, s_red, s_cand, s_src);
  }
  if (tid < kc) {
    const unsigned long long key = s_cand[tid];
    s_sim[tid] = key ? f32_unordered((uint32_t)(key >> 32)) : -INFINITY;
    s_idx[tid] = key ? (int32_t)(0xffffffffu - (uint32_t)key) : -1;
  }
  __syncthreads();

  // labels of all kc candidates are requested before the re-rank and parked after it (independent gathers); the
  // threads are rotated by half a block so that, for the usual handful of candidates, the label gathers are issued
  // by the upper warps while the lower ones (warp c = candidate c) already fetch their bank rows
  const int tid_lab = (tid + (kFinThreads >> 1)) & (kFinThreads - 1);   // the block size is a power of two
  float lv[4];
  const int nlab = kc * 2 * M;   // <= 64 * 32 = 4 * 512
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int e = tid_lab + u * kFinThreads;
    lv[u] = 0.0f;
    if (e < nlab) {
      const int c = e / (2 * M), col = e - c * 2 * M;
      const int32_t id = s_idx[c];
      if (id >= 0) lv[u] = (col < M) ? a.bank_quality[(size_t)id * M + col] : a.bank_outlen[(size_t)id * M + col - M];
    }
  }
  // ---- exact re-rank ----
  if (a.rerank) {
    for (int c = warp; c < kc; c += nwarps) {
      const int32_t id = s_idx[c];
      if (id < 0) continue;
      const float sx = exact_sim_bf16(qrow, reinterpret_cast<const uint4*>(a.bank + (size_t)id * a.d), nvec, lane);
      if (lane == 0) s_sim[c] = sx;
    }
    __syncthreads();
  }
  // rank by counting (keys are distinct because indices are): warp c ranks candidate c, lane j compares candidate j
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
    if (lane == 0) {
      o_sim[rank] = sc;
      o_idx[rank] = id;
      o_pos[rank] = c;
      if (rank < k) {   // ---- weight of the rank-th neighbour (the warps' square roots and divisions overlap) ----
        float w = 1.0f;
        if (id < 0) {
          w = 0.0f;   // fewer than k rows reachable (cannot happen for k <= N); keeps the gather in bounds
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
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int e = tid_lab + u * kFinThreads;
    if (e < nlab) s_lab[e / (2 * M)][e % (2 * M)] = lv[u];
  }
  __syncthreads();
  // ---- aggregate: thread m < M -> quality, M <= thread < 2M -> output length ----
  if (tid < 2 * M) {
    const int m = tid % M;
    float num = 0.0f, den = 0.0f;
    // (a missing neighbour -- fewer than k rows reachable -- has weight 0 and position 0: it adds +0 to both sums)
#pragma unroll 4   // the loads of four neighbours in flight; the two sums stay sequential (canonical order)
    for (int j = 0; j < k; ++j) {
      const float w = s_w[j];
      const float p = __fmul_rn(w, s_lab[o_pos[j]][tid]);
      num = __fadd_rn(num, p);
      den = __fadd_rn(den, w);
    }
    const float pred = __fdiv_rn(num, den);
    if (tid < M) {
      sQ[m] = pred;
      a.pred_q[(size_t)r * M + m] = pred;
      if (out_pq) out_pq[(size_t)r * M + m] = pred;
    } else {
      sL[m] = pred;
      a.pred_l[(size_t)r * M + m] = pred;
      if (out_pl) out_pl[(size_t)r * M + m] = pred;
    }
  }
  if (!a.with_terms || warp != 0) return;
  // ---- per-(request, tier) terms: warp 0 alone (2M <= 32: the predictions above were all written by its lanes) ----
  const uint32_t present = __ballot_sync(0xffffffffu, c_present != 0);   // lanes 0..M-1 hold the tiers' flags
  __syncwarp();
  {
    const int m = lane < M ? lane : 0;
    const float L = sL[m];
    const float C = __fadd_rn(__fmul_rn(c_ell, c_pin), __fmul_rn(L, c_pout));
    float kmax;
    const float A = tier_term_A_warp(lane, present, C, L, sQ[m], c_wq, c_wc, has_budget, c_budget, &kmax);
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
  // keys of all lists + the warps' merged lists (keys and sources); the rescan's second merge reuses the front
  const size_t n1 = (size_t)nlists * kcap * 8 + (size_t)kFinWarpsMax * kMerge2Stride * 12;
  const size_t n2 = (size_t)(kFinWarpsMax + 1) * kMerge2Stride * 8;
  return n1 > n2 ? n1 : n2;
}

cudaError_t finish_prepare(size_t max_smem) {
  return cudaFuncSetAttribute(finish_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem);
}

cudaError_t launch_finish(const FinishArgs& a, InstTable t, const CallParams& cp, int B, cudaStream_t s) {
  // 32 warps from 257 lists on: the first-level merges' admission bound needs at least k + slack warps to bite
  const cudaError_t e = launch_chained(finish_kernel, dim3(B), dim3(a.nlists > 256 ? 1024 : 512),
                                       finish_smem_bytes(a.nlists, a.kcap), s, a, t, cp);
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rb
