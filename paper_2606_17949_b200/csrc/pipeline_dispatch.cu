// pipeline_dispatch.cu -- pipeline-mode dispatchers: "Equation 1 is bypassed, a pluggable estimator first picks
// a model ..., and a dispatcher (round-robin, shortest-queue, or random) places the request within that model's replica
// pool."  The model per request is an input; the three dispatchers run here, in input order, over the dead-reckoned state
// and with the greedy pass's update (d += L^, b = min(b+1, cap); reading 18):
//   policy 0  round-robin: the tier's instances in index order, one cursor per tier that persists across batches
//   policy 1  shortest queue: the tier's instance with the smallest d, ties -> smaller index
//   policy 2  random: member splitmix64(seed + counter) mod n of the tier's instances; counter = requests placed so far
// One warp; the state lives in shared memory; the members of a tier are a contiguous run of `members` (instances sorted
// by (tier, index), built by rb_set_instances).
#include "rb_internal.cuh"

namespace rb {
namespace {

__device__ __forceinline__ unsigned long long splitmix64(unsigned long long x) {
  x += 0x9e3779b97f4a7c15ull;
  x = (x ^ (x >> 30)) * 0xbf58476d1ce4e5b9ull;
  x = (x ^ (x >> 27)) * 0x94d049bb133111ebull;
  return x ^ (x >> 31);
}

__global__ void __launch_bounds__(32)
pipeline_dispatch_kernel(InstTable t, const int32_t* __restrict__ members, const int32_t* __restrict__ tstart,
                         float* __restrict__ dq, int32_t* __restrict__ bq, const int32_t* __restrict__ model,
                         const float* __restrict__ outlen, int B, int policy, unsigned long long seed,
                         unsigned long long* __restrict__ counter, int32_t* __restrict__ cursor, int commit,
                         int32_t* __restrict__ assignment) {
  __shared__ float s_d[kMaxI];
  __shared__ int32_t s_b[kMaxI];
  __shared__ int32_t s_cur[kMaxM];
  const int lane = threadIdx.x, I = t.I, M = t.M;
  for (int i = lane; i < I; i += 32) { s_d[i] = dq[i]; s_b[i] = bq[i]; }
  if (lane < M) s_cur[lane] = cursor[lane];
  unsigned long long cnt = *counter;
  __syncwarp();
  for (int r = 0; r < B; ++r) {
    const int m = model[r];
    int pick = -1;
    if (m >= 0 && m < M) {
      const int s0 = tstart[m], n = tstart[m + 1] - s0;
      if (n > 0) {
        if (policy == 0) {
          const int c = s_cur[m];
          pick = members[s0 + c % n];
          __syncwarp();
          if (lane == 0) s_cur[m] = (c + 1) % n;
        } else if (policy == 2) {
          pick = members[s0 + (int)(splitmix64(seed + cnt) % (unsigned long long)n)];
        } else {
          uint32_t bd = 0xffffffffu;
          int bi = 0x7fffffff;
          for (int j = lane; j < n; j += 32) {
            const int i = members[s0 + j];
            const uint32_t dk = __float_as_uint(__fadd_rn(s_d[i], 0.0f));   // d >= 0: bit order == float order
            if (dk < bd) { bd = dk; bi = i; }                              // members ascend: ties keep the smaller i
          }
          const uint32_t gd = __reduce_min_sync(0xffffffffu, bd);
          pick = (int)__reduce_min_sync(0xffffffffu, bd == gd ? (uint32_t)bi : 0xffffffffu);
        }
        ++cnt;
        if (outlen != nullptr && lane == 0) {
          s_d[pick] = __fadd_rn(s_d[pick], outlen[(size_t)r * M + m]);
          if (s_b[pick] < t.cap[pick]) s_b[pick] += 1;
        }
      }
    }
    if (lane == 0) assignment[r] = pick;
    __syncwarp();
  }
  if (commit) {
    if (outlen != nullptr)
      for (int i = lane; i < I; i += 32) { dq[i] = s_d[i]; bq[i] = s_b[i]; }
    if (lane < M) cursor[lane] = s_cur[lane];
    if (lane == 0) *counter = cnt;
  }
}

}  // namespace

cudaError_t launch_pipeline_dispatch(InstTable t, const int32_t* members, const int32_t* tstart, float* dq, int32_t* bq,
                                     const int32_t* model, const float* outlen, int B, int policy, unsigned long long seed,
                                     unsigned long long* counter, int32_t* cursor, int commit, int32_t* assignment,
                                     cudaStream_t s) {
  pipeline_dispatch_kernel<<<1, 32, 0, s>>>(t, members, tstart, dq, bq, model, outlen, B, policy, seed, counter, cursor, commit,
                                            assignment);
  return cudaGetLastError();
}

}  // namespace rb
