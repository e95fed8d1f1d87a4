// match_replay.cu -- batch-level matching replay.
//
// "A batch-level matching (e.g. Hungarian) would differ only through within-batch state updates, and an offline
// replay over the logged score matrices changes 15.6% of assignments ...".  Given the batch-start score matrix
// S0 [B x I] (rb_decide_from_predictions' scores0; -inf = filtered out by the request's budget) and a quota of requests
// per instance, the kernel finds the assignment a maximising sum_r S0[r, a(r)] with at most quota[i] requests on
// instance i (reading 26), and counts how many requests it places differently from a given (greedy)
// assignment.
//
// Method: the Hungarian method in its shortest-augmenting-path form (Jonker-Volgenant) on the transportation form of
// the problem -- requests are inserted one by one; each insertion is a Dijkstra search over the INSTANCES (columns) in
// reduced costs c[r][i] - u[r] - v[i], where a full instance passes the search on through every request it holds; the
// search ends at the first instance with a free slot, the dual variables u, v are updated so that reduced costs stay
// non-negative and assigned pairs tight, and the path is flipped.  One CTA; thread i owns column i (dist, v, load);
// per search step one block-wide argmin and one relaxation sweep per request of the scanned column.  Arithmetic in
// fp64 on the fp32 scores: the optimum's objective is compared with the oracle's (the optimal assignment itself need
// not be unique).
#include "rb_internal.cuh"

namespace rb {
namespace {

constexpr int kMatchThreads = 1024;   // >= kMaxI: one column per thread

struct MinPair { double v; int i; };

__device__ __forceinline__ MinPair warp_argmin(double v, int i) {
  for (int o = 16; o > 0; o >>= 1) {
    const double ov = __shfl_xor_sync(0xffffffffu, v, o);
    const int oi = __shfl_xor_sync(0xffffffffu, i, o);
    if (ov < v || (ov == v && oi < i)) { v = ov; i = oi; }
  }
  return MinPair{v, i};
}

// status: 0 ok, 1 infeasible (some request has no admissible instance with room left along any path)
__global__ void __launch_bounds__(kMatchThreads)
match_replay_kernel(const float* __restrict__ S0, int B, int I, const int32_t* __restrict__ quota,
                    const int32_t* __restrict__ greedy, int32_t* __restrict__ match, double* __restrict__ objective,
                    int32_t* __restrict__ n_diverged, int32_t* __restrict__ status) {
  extern __shared__ unsigned char smem_raw[];
  double* u = reinterpret_cast<double*>(smem_raw);          // [B] row duals
  int32_t* asg = reinterpret_cast<int32_t*>(u + B);         // [B] column of row r, -1 = not inserted yet
  int32_t* nxt = asg + B;                                   // [B] next row in the same column's list
  int32_t* head = nxt + B;                                  // [I] first row of column i, -1 = none
  int32_t* pred = head + I;                                 // [I] row through which column i was reached
  __shared__ double s_rv[32];
  __shared__ int s_ri[32];
  __shared__ double s_delta;
  __shared__ int s_sink, s_fail, s_free;
  const int i = threadIdx.x, lane = i & 31, warp = i >> 5, nwarps = blockDim.x >> 5;
  const bool col = i < I;
  double v = 0.0;                       // column dual
  int load = 0;
  const int cap = col ? quota[i] : 0;
  for (int r = i; r < B; r += blockDim.x) { u[r] = 0.0; asg[r] = -1; nxt[r] = -1; }
  if (col) head[i] = -1;
  if (i == 0) s_fail = 0;
  __syncthreads();

  for (int r0 = 0; r0 < B && !s_fail; ++r0) {
    // ---- Dijkstra over columns from the new row r0 ----
    double dist = INFINITY;
    bool scanned = false;
    if (col) {
      const float s = S0[(size_t)r0 * I + i];
      dist = (s == -INFINITY) ? INFINITY : (-(double)s - u[r0] - v);
      pred[i] = r0;
    }
    int sink = -1;
    double delta = 0.0;
    while (true) {
      // block argmin of dist over unscanned columns
      MinPair m = warp_argmin((col && !scanned) ? dist : INFINITY, i);
      if (lane == 0) { s_rv[warp] = m.v; s_ri[warp] = m.i; }
      __syncthreads();
      if (warp == 0) {
        MinPair g = warp_argmin(lane < nwarps ? s_rv[lane] : INFINITY, lane < nwarps ? s_ri[lane] : 0x7fffffff);
        if (lane == 0) { s_delta = g.v; s_sink = g.i; }
      }
      __syncthreads();
      const double dj = s_delta;
      const int j = s_sink;
      if (!(dj < INFINITY)) { sink = -1; break; }      // nothing reachable: infeasible
      if (i == j) s_free = (load < cap) ? 1 : 0;
      __syncthreads();
      if (s_free) { sink = j; delta = dj; break; }
      // column j is full: scan it -- the search continues through every row it holds
      if (i == j) scanned = true;
      for (int r = head[j]; r >= 0; r = nxt[r]) {
        if (col && !scanned) {
          const float s = S0[(size_t)r * I + i];
          if (s != -INFINITY) {
            const double nd = dj + (-(double)s - u[r] - v);
            if (nd < dist) { dist = nd; pred[i] = r; }
          }
        }
      }
      __syncthreads();   // s_delta / s_sink / s_free are rewritten in the next round
    }
    if (sink < 0) {
      if (i == 0) s_fail = 1;
      __syncthreads();
      break;
    }
    // ---- dual update: scanned columns and the rows they hold move by (delta - dist[column]); r0 by delta ----
    if (col && scanned) {
      const double shift = delta - dist;
      for (int r = head[i]; r >= 0; r = nxt[r]) u[r] += shift;
      v -= shift;
    }
    if (i == 0) u[r0] += delta;
    __syncthreads();
    // ---- flip the path: sink <- pred row <- its old column <- ... <- r0 ----
    if (i == 0) {
      int jcol = sink;
      while (true) {
        const int r = pred[jcol];
        const int old = asg[r];
        // unlink r from its old column
        if (old >= 0) {
          int p = head[old];
          if (p == r) head[old] = nxt[r];
          else { while (nxt[p] != r) p = nxt[p]; nxt[p] = nxt[r]; }
        }
        asg[r] = jcol;
        nxt[r] = head[jcol];
        head[jcol] = r;
        if (r == r0) break;
        jcol = old;
      }
    }
    __syncthreads();
    if (i == sink) load += 1;      // every other column on the path loses one row and gains one
    __syncthreads();
  }

  // ---- outputs ----
  if (i == 0) *status = s_fail;
  if (s_fail) return;
  double part = 0.0;
  int div = 0;
  for (int r = i; r < B; r += blockDim.x) {
    const int a = asg[r];
    match[r] = a;
    part += (double)S0[(size_t)r * I + a];
    if (greedy != nullptr) div += (greedy[r] != a);
  }
  for (int o = 16; o > 0; o >>= 1) {
    part += __shfl_xor_sync(0xffffffffu, part, o);
    div += __shfl_xor_sync(0xffffffffu, div, o);
  }
  __syncthreads();
  if (lane == 0) { s_rv[warp] = part; s_ri[warp] = div; }
  __syncthreads();
  if (i == 0) {
    double t = 0.0;
    int dsum = 0;
    for (int w = 0; w < nwarps; ++w) { t += s_rv[w]; dsum += s_ri[w]; }
    *objective = t;
    *n_diverged = dsum;
  }
}

}  // namespace

cudaError_t match_replay_prepare() {
  return cudaFuncSetAttribute(match_replay_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}

cudaError_t launch_match_replay(const float* S0, int B, int I, const int32_t* quota, const int32_t* greedy, int32_t* match,
                                double* objective, int32_t* n_diverged, int32_t* status, cudaStream_t s) {
  const size_t smem = (size_t)B * (8 + 4 + 4) + (size_t)I * 8;
  match_replay_kernel<<<1, kMatchThreads, smem, s>>>(S0, B, I, quota, greedy, match, objective, n_diverged, status);
  return cudaGetLastError();
}

}  // namespace rb
