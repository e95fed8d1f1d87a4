// estimate.cu -- the estimate stage around the tensor-core scan: query staging (a0), the exact fp32-storage
// scan (a1, small banks), the cross-CTA top-k merge (a2) and the re-rank + aggregate kernel (a3).
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
__device__ __forceinline__ unsigned long long shfl64(unsigned long long x, int src) {
  return __shfl_sync(0xffffffffu, x, src);
}
__device__ __forceinline__ unsigned long long shfl64_up1(unsigned long long x) { return __shfl_up_sync(0xffffffffu, x, 1); }

// ---- a0 ---------------------------------------------------------------------------------------------
__global__ void stage_queries_kernel(const float* __restrict__ q, __nv_bfloat16* __restrict__ qs, int B, int Bpad, int d) {
  const size_t n = (size_t)Bpad * d;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t r = i / d;
    qs[i] = (r < (size_t)B) ? __float2bfloat16_rn(q[i]) : __float2bfloat16_rn(0.0f);
  }
}

// ---- a1, fp32 storage -----------------------------------------------------------------------------------
// s[r,n] = fl32( sum_c (double)x[r,c] * (double)e[n,c] ) in index order: the product of two fp32 values is
// exact in fp64, so one fp64 FMA per term is exactly "multiply, then add with one rounding".
constexpr int kF32Rows = 128;   // bank rows per block, one per thread
constexpr int kF32Q = 8;        // queries per register group
constexpr int kF32Chunk = 64;   // columns staged per step
__global__ void __launch_bounds__(kF32Rows)
scan_f32_kernel(const float* __restrict__ bank, const float* __restrict__ q, int64_t N, int d, int nq, float* __restrict__ sims) {
  __shared__ float xs[kF32Q][kF32Chunk];
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

// ---- a2 ---------------------------------------------------------------------------------------------
// One warp per query.  The running best-kc list lives across the warp (rank l in lane l, rank 32+l in the
// second register); candidates stream in 32 at a time, survivors of the threshold are inserted one by one
// with ballots and shuffles.  part_* layout: [grid][kcap][Bpad].
__global__ void __launch_bounds__(128)
merge_kernel(const float* __restrict__ part_sim, const int32_t* __restrict__ part_idx, int grid, int kcap, int Bpad, int B,
             int kc, int64_t N, float* __restrict__ cand_sim, int32_t* __restrict__ cand_idx) {
  const int r = blockIdx.x * 4 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (r >= B) return;
  unsigned long long a = 0, b = 0;   // ranks lane and 32+lane, descending
  unsigned long long thr = 0;        // key of rank kc-1
  const int total = grid * kcap;
  for (int base = 0; base < total; base += 32) {
    const int e = base + lane;
    unsigned long long key = 0;
    if (e < total) {
      const size_t off = (size_t)e * Bpad + r;
      const int32_t id = part_idx[off];
      if (id >= 0 && (int64_t)id < N) key = make_key(part_sim[off], id);
    }
    unsigned mask = __ballot_sync(0xffffffffu, key > thr);
    while (mask) {
      const int src = __ffs(mask) - 1;
      mask &= mask - 1;
      const unsigned long long x = shfl64(key, src);
      if (x > thr) {
        const int p = __popc(__ballot_sync(0xffffffffu, a > x)) + __popc(__ballot_sync(0xffffffffu, b > x));
        const unsigned long long a_up = shfl64_up1(a), b_up = shfl64_up1(b), a_last = shfl64(a, 31);
        const unsigned long long b_prev = (lane == 0) ? a_last : b_up;
        a = (lane < p) ? a : ((lane == p) ? x : a_up);
        b = (lane + 32 < p) ? b : ((lane + 32 == p) ? x : b_prev);
        thr = (kc <= 32) ? shfl64(a, kc - 1) : shfl64(b, kc - 33);
      }
    }
  }
  for (int j = lane; j < kc; j += 32) {
    const unsigned long long key = (j < 32) ? a : b;
    const size_t o = (size_t)r * kc + j;
    if (key == 0) {
      cand_sim[o] = -INFINITY;
      cand_idx[o] = -1;
    } else {
      cand_sim[o] = f32_unordered((uint32_t)(key >> 32));
      cand_idx[o] = (int32_t)(0xffffffffu - (uint32_t)key);
    }
  }
}

// ---- a3 ---------------------------------------------------------------------------------------------
// One block per query.  Optional exact re-rank (bf16 storage): the kc candidates' similarities are recomputed
// from the stored bf16 rows with fp64 accumulation (products of bf16 values are exact), rounded once to fp32,
// and re-ordered by (s desc, n asc); the best k are the neighbours.  Then:
//   t = 2*s; u = 2 - t; u = max(u,0); dist = sqrt(u); w = 1/(dist + eps)      (uniform mode: w = 1)
//   num_m = sum_j w_j*label[n_j,m] (j ascending, multiply then add); den = sum_j w_j; pred = num/den
constexpr int kAggThreads = 256;
__global__ void __launch_bounds__(kAggThreads)
aggregate_kernel(const __nv_bfloat16* __restrict__ bank, const __nv_bfloat16* __restrict__ qs, int d, int rerank,
                 const float* __restrict__ cand_sim, const int32_t* __restrict__ cand_idx, int kc, int k,
                 const float* __restrict__ bank_quality, const float* __restrict__ bank_outlen, int M, int weight_mode,
                 float eps, int32_t* __restrict__ nn_idx, float* __restrict__ nn_sim, float* __restrict__ pred_q,
                 float* __restrict__ pred_l) {
  __shared__ float s_sim[kMaxK];
  __shared__ int32_t s_idx[kMaxK];
  __shared__ float o_sim[kMaxK];
  __shared__ int32_t o_idx[kMaxK];
  __shared__ float s_w[kMaxK];
  const int r = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = kAggThreads / 32;
  if (threadIdx.x < kc) {
    s_sim[threadIdx.x] = cand_sim[(size_t)r * kc + threadIdx.x];
    s_idx[threadIdx.x] = cand_idx[(size_t)r * kc + threadIdx.x];
  }
  __syncthreads();
  if (rerank) {
    const uint4* qrow = reinterpret_cast<const uint4*>(qs + (size_t)r * d);
    const int nvec = d / 8;   // d % 8 == 0
    for (int c = warp; c < kc; c += nwarps) {
      const int32_t id = s_idx[c];
      if (id < 0) continue;
      const uint4* brow = reinterpret_cast<const uint4*>(bank + (size_t)id * d);
      double acc = 0.0;
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
      if (lane == 0) s_sim[c] = (float)acc;
    }
    __syncthreads();
  }
  // rank by counting (keys are distinct because indices are)
  if (threadIdx.x < kc) {
    const int32_t id = s_idx[threadIdx.x];
    const unsigned long long me = (id < 0) ? 0ull : make_key(s_sim[threadIdx.x], id);
    int rank = 0;
    for (int j = 0; j < kc; ++j) {
      const int32_t oj = s_idx[j];
      const unsigned long long other = (oj < 0) ? 0ull : make_key(s_sim[j], oj);
      rank += (other > me) || (other == me && j < (int)threadIdx.x);
    }
    o_sim[rank] = s_sim[threadIdx.x];
    o_idx[rank] = id;
  }
  __syncthreads();
  if (threadIdx.x < k) {
    const float s = o_sim[threadIdx.x];
    float w = 1.0f;
    if (o_idx[threadIdx.x] < 0) {
      w = 0.0f;   // fewer than k rows reachable (cannot happen for k <= N); keeps the gather in bounds
    } else if (weight_mode == 0) {
      const float t = __fmul_rn(2.0f, s);
      float u = __fsub_rn(2.0f, t);
      u = fmaxf(u, 0.0f);
      const float dist = __fsqrt_rn(u);
      w = __fdiv_rn(1.0f, __fadd_rn(dist, eps));
    }
    s_w[threadIdx.x] = w;
    if (nn_idx) nn_idx[(size_t)r * k + threadIdx.x] = o_idx[threadIdx.x];
    if (nn_sim) nn_sim[(size_t)r * k + threadIdx.x] = s;
  }
  __syncthreads();
  if (threadIdx.x < 2 * M) {
    const int m = threadIdx.x % M;
    const float* lab = (threadIdx.x < M) ? bank_quality : bank_outlen;
    float num = 0.0f, den = 0.0f;
    for (int j = 0; j < k; ++j) {
      const float w = s_w[j];
      if (o_idx[j] < 0) continue;
      const float p = __fmul_rn(w, lab[(size_t)o_idx[j] * M + m]);
      num = __fadd_rn(num, p);
      den = __fadd_rn(den, w);
    }
    const float pred = __fdiv_rn(num, den);
    if (threadIdx.x < M) pred_q[(size_t)r * M + m] = pred;
    else pred_l[(size_t)r * M + m] = pred;
  }
}

}  // namespace

cudaError_t launch_stage_queries(const float* q, __nv_bfloat16* qs, int B, int Bpad, int d, cudaStream_t s) {
  const size_t n = (size_t)Bpad * d;
  int blocks = (int)((n + 255) / 256);
  if (blocks > 148 * 8) blocks = 148 * 8;
  stage_queries_kernel<<<blocks, 256, 0, s>>>(q, qs, B, Bpad, d);
  return cudaGetLastError();
}

cudaError_t launch_scan_f32(const float* bank, const float* q, int64_t N, int d, int nq, float* sims, cudaStream_t s) {
  const int blocks = (int)((N + kF32Rows - 1) / kF32Rows);
  scan_f32_kernel<<<blocks, kF32Rows, 0, s>>>(bank, q, N, d, nq, sims);
  return cudaGetLastError();
}

cudaError_t launch_select_f32(const float* sims, int64_t N, int nq, int kc, float* cand_sim, int32_t* cand_idx,
                              cudaStream_t s) {
  select_f32_kernel<<<nq, 256, 0, s>>>(sims, N, kc, cand_sim, cand_idx);
  return cudaGetLastError();
}

cudaError_t launch_merge(const float* part_sim, const int32_t* part_idx, int grid, int kcap, int Bpad, int B, int kc,
                         int64_t N, float* cand_sim, int32_t* cand_idx, cudaStream_t s) {
  merge_kernel<<<(B + 3) / 4, 128, 0, s>>>(part_sim, part_idx, grid, kcap, Bpad, B, kc, N, cand_sim, cand_idx);
  return cudaGetLastError();
}

cudaError_t launch_aggregate(const __nv_bfloat16* bank, const __nv_bfloat16* qs, int d, int rerank, const float* cand_sim,
                             const int32_t* cand_idx, int kc, int k, const float* bank_quality, const float* bank_outlen,
                             int M, int weight_mode, float eps, int B, int32_t* nn_idx, float* nn_sim, float* pred_q,
                             float* pred_l, cudaStream_t s) {
  aggregate_kernel<<<B, kAggThreads, 0, s>>>(bank, qs, d, rerank, cand_sim, cand_idx, kc, k, bank_quality, bank_outlen, M,
                                             weight_mode, eps, nn_idx, nn_sim, pred_q, pred_l);
  return cudaGetLastError();
}

}  // namespace rb
