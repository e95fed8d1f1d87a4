// scan_tc2.cu -- step a1 for bf16 storage and large batches (B > 128, the tensor-bound regime): the same
// similarity scan with fused per-query top-KCAP as scan_tc.cu, on CTA PAIRS (tcgen05 cta_group::2).
//
// Definition (readings 1, 3, 4): s[r,n] = <q~_r, e~_n> over the bf16-rounded vectors; per
// (query, slab of bank rows) the best KCAP entries in the order (s descending, n ascending).
//
// Why pairs: with one CTA per SM a 128 x 256 x 64 step moves 48 KB of operands from L2 per 512 tensor-pipe
// clocks (96 B/clk/SM), and the L2 -> SM fabric, not the tensor pipe, bounds the kernel (measured 1.0 PFLOP/s
// = 11.8 TB/s of TMA fill).  A pair computes a 256 x 256 tile: each CTA stages its own 128 queries and HALF of
// the bank tile (128 rows), the MMA reads both halves, so the same 512 clocks need 32 KB per SM.
//
// Shape: grid = 2 x 74 (one cluster per TPC), 6 warps per CTA.
//   warp 0   TMA producer (both CTAs): own 128 queries + own 128 bank rows per K chunk into a 6-stage ring; the
//            bytes of both CTAs complete on the LEADER's (rank 0) "full" barrier.
//   warp 1   TMEM allocation (512 columns, cta_group::2, both CTAs); lane 0 of the leader issues the MMAs
//            (M = 256 = 2 x 128 queries, N = 256 bank rows, K = 16) and commits to both CTAs' barriers.
//   warps 2-5  epilogue (both CTAs): thread t = TMEM lane t = query (m-pair * 256 + rank * 128 + t), all 256
//            columns of the accumulator.
// A cluster owns a contiguous slab of whole 256-row tiles and visits every m-pair per tile (the bank tile comes
// from L2 after the first visit).  The per-(slab, query) lists live in global memory (L2); a visit needs only
// the admission threshold (shared memory) and touches the list itself only when a candidate beats it.
// Thresholds are shared ACROSS slabs: a slab that has K = KCAP >= k + slack entries for a query publishes its
// K-th best similarity (atomicMax on gthr[query]); that value bounds the query's global K-th best from below, so
// every slab may drop what is strictly below it without changing the merged result.  This turns the
// K ln(rows per slab) insertions per (slab, query) of independent streaming top-K lists into about
// K ln(rows seen by all slabs together) per query, which keeps the epilogue off the tensor pipe's time line.
#include "rb_internal.cuh"
#include "tc_scan.cuh"

namespace rb {
namespace {


constexpr int kStages2 = 6;
constexpr int kA2Bytes = kTileM * kTileK * 2;            // 16 KB: this CTA's 128 queries x 64 bf16
constexpr int kB2Bytes = (kTileN / 2) * kTileK * 2;      // 16 KB: this CTA's 128 of the tile's 256 bank rows
constexpr int kStage2Bytes = kA2Bytes + kB2Bytes;        // 32 KB
constexpr int kThreads2 = 256;                            // 6 pipeline warps + 2 bound refreshers
constexpr int kCand2Slots = 16;                           // parked survivors per thread
constexpr int kMaxPairs = 16;                             // m-pairs of one decision: B <= 4096
constexpr int kSmem2Bytes = kStages2 * kStage2Bytes + kCand2Slots * kTileM * 8 + 2 * kMaxPairs * kTileM * 4 + 256 + 1024;
constexpr int kPairM = 2 * kTileM;                        // queries per m-pair

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same variable in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
  return r;
}
// Arrive on a barrier of another CTA of the cluster.  Relaxed: what the arrival publishes is that this warp's
// tcgen05.ld reads of the accumulator have completed (tcgen05.wait::ld + tcgen05.fence::before_thread_sync order
// them before it); no ordinary memory is handed over, and a release at cluster scope costs ~1500 clocks per visit.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// TMA tile load of a CTA pair: data into this CTA's shared memory, bytes counted on the barrier at bar_cluster_addr
// (the leader's).
__device__ __forceinline__ void tma_load_2d_pair(void* dst, const CUtensorMap* map, int c0, int c1, uint32_t bar_cluster_addr) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(bar_cluster_addr)
      : "memory");
}
__device__ __forceinline__ void tc_commit_pair(uint64_t* bar) {   // arrives on this barrier in BOTH CTAs of the pair
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                   smem_u32(bar)),
               "h"((uint16_t)3)
               : "memory");
}
// D[tmem, both CTAs] (+)= A * B^T: 256 x N x 16, each CTA supplying 128 rows of A and N/2 rows of B.
__device__ __forceinline__ void tc_mma_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum)
      : "memory");
}

// Per-thread state of one visit (one accumulator of one m-pair): the admission threshold, the survivors parked
// in shared memory, and the thread's list, which is fetched from global memory when the first survivor appears
// and consumed only when the survivors are inserted -- normally after the accumulator has been released, so that
// neither the L2 round trip nor the insertion sits on the tensor pipe's time line.
template <int K>
struct Visit {
  float v[K];
  int32_t ix[K];
  float thr;
  int cnt;        // survivors parked
  bool loaded;    // list requested (or initialised)
};

// Inserts the parked survivors (scan order) into the list, in warp lock-step: every lane inserts its p-th
// survivor in the same iteration.
template <int K>
__device__ __forceinline__ void request_list(Visit<K>& st, const float4* ps4, const int4* pi4) {
  if (st.cnt > 0 && !st.loaded) {
#pragma unroll
    for (int j = 0; j < K / 4; ++j) {
      const float4 a = ps4[j];
      const int4 b = pi4[j];
      st.v[4 * j] = a.x; st.v[4 * j + 1] = a.y; st.v[4 * j + 2] = a.z; st.v[4 * j + 3] = a.w;
      st.ix[4 * j] = b.x; st.ix[4 * j + 1] = b.y; st.ix[4 * j + 2] = b.z; st.ix[4 * j + 3] = b.w;
    }
    st.loaded = true;
  }
}
template <int K>
__device__ __forceinline__ void drain(Visit<K>& st, const float4* ps4, const int4* pi4, const uint2* cand, int tl, int n0) {
  request_list<K>(st, ps4, pi4);
  uint2 nxt = cand[tl];
  for (int p = 0; __any_sync(0xffffffffu, p < st.cnt); ++p) {
    const uint2 cur = nxt;
    nxt = cand[min(p + 1, kCand2Slots - 1) * kTileM + tl];
    const float s = __uint_as_float(cur.x);
    if (p < st.cnt && s > st.thr) {
      list_insert<K>(st.v, st.ix, s, n0 + (int)cur.y);
      st.thr = fmaxf(st.thr, st.v[K - 1]);
    }
  }
  st.cnt = 0;
}

// One tcgen05.ld chunk (32 similarities of this thread's query against bank rows n0 + c0 ..).  Steady state: no
// lane of the warp holds a similarity above its threshold: one max tree and one vote.  Otherwise the survivors
// are parked, 8 columns at a time; the queue (kCand2Slots per thread) is drained early only when a lane could
// overflow it, which happens in the first tiles of a slab, while the lists fill.
template <int K>
__device__ __forceinline__ void park_chunk(const uint32_t (&regs)[32], int c0, int c_end, int n0, Visit<K>& st,
                                           const float4* ps4, const int4* pi4, uint2* cand, int tl) {
  const bool full = c0 + 32 <= c_end;   // warp-uniform
  float m0 = -INFINITY, m1 = -INFINITY, m2 = -INFINITY, m3 = -INFINITY;
  if (full) {
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
      m0 = fmaxf(m0, __uint_as_float(regs[j + 0]));
      m1 = fmaxf(m1, __uint_as_float(regs[j + 1]));
      m2 = fmaxf(m2, __uint_as_float(regs[j + 2]));
      m3 = fmaxf(m3, __uint_as_float(regs[j + 3]));
    }
  } else {
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
      m0 = fmaxf(m0, (c0 + j + 0 < c_end) ? __uint_as_float(regs[j + 0]) : -INFINITY);
      m1 = fmaxf(m1, (c0 + j + 1 < c_end) ? __uint_as_float(regs[j + 1]) : -INFINITY);
      m2 = fmaxf(m2, (c0 + j + 2 < c_end) ? __uint_as_float(regs[j + 2]) : -INFINITY);
      m3 = fmaxf(m3, (c0 + j + 3 < c_end) ? __uint_as_float(regs[j + 3]) : -INFINITY);
    }
  }
  const float m = fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
  if (!__any_sync(0xffffffffu, m > st.thr)) return;
#pragma unroll
  for (int g = 0; g < 4; ++g) {
    if (__any_sync(0xffffffffu, st.cnt > kCand2Slots - 8)) drain<K>(st, ps4, pi4, cand, tl, n0);
#pragma unroll
    for (int j = 8 * g; j < 8 * g + 8; ++j) {
      const float s = __uint_as_float(regs[j]);
      if ((full || c0 + j < c_end) && s > st.thr) {
        cand[st.cnt * kTileM + tl] = make_uint2(regs[j], (uint32_t)(c0 + j));
        ++st.cnt;
      }
    }
  }
  request_list<K>(st, ps4, pi4);   // nothing waits for it here
}

template <int KCAP>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads2, 1)
scan_tc2_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_bank, int64_t N, int d,
                int B, int Bpad, float* part_sim, int32_t* part_idx, uint32_t* gthr, int pub_j, int pub_groups,
                int publish_own) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint2* cand = (uint2*)(smem + kStages2 * kStage2Bytes);
  float* thr_s = (float*)(cand + kCand2Slots * kTileM);   // [n_mp][128] K-th best similarity of this CTA's lists
  uint32_t* gl_s = (uint32_t*)(thr_s + kMaxPairs * kTileM);   // [n_mp][128] pooled lower bound (ordered), see refresh
  uint64_t* bars = (uint64_t*)(gl_s + kMaxPairs * kTileM);
  uint64_t* full = bars;                   // [kStages2] leader's: both CTAs' TMA bytes landed
  uint64_t* empty = bars + kStages2;       // [kStages2] own: the MMAs that read the slot retired
  uint64_t* tfull = bars + 2 * kStages2;   // [2] own: accumulator complete
  uint64_t* tempty = tfull + 2;            // [2] leader's: accumulator drained by the 8 epilogue warps of the pair
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);
  int* epi_done = (int*)(tmem_slot + 1);   // epilogue warps that have finished

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cl = blockIdx.x >> 1, ncl = gridDim.x >> 1;
  const int n_mp = Bpad / kPairM;
  const int nk = (d + kTileK - 1) / kTileK;
  const int64_t tiles_total = (N + kTileN - 1) / kTileN;
  const int64_t t0 = tiles_total * cl / ncl, t1 = tiles_total * (cl + 1) / ncl;
  const int ntiles = (int)(t1 - t0);
  const int64_t row0 = t0 * kTileN;

  launch_dependents();
  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_q) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_bank) : "memory");
    for (int s = 0; s < kStages2; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&tfull[a], 1);
      mbar_init(&tempty[a], 8);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (threadIdx.x == 32) *epi_done = 0;
  for (int i = threadIdx.x; i < kMaxPairs * kTileM; i += kThreads2) gl_s[i] = 0u;
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  cluster_sync_all();   // barriers of both CTAs initialised, TMEM allocated in both
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer (both CTAs) =====
    if (lane == 0) {
      grid_dependency_wait();   // the staged queries come from the preceding kernel
      uint32_t full_leader[kStages2];
#pragma unroll
      for (int s = 0; s < kStages2; ++s) full_leader[s] = mapa_u32(smem_u32(&full[s]), 0);
      uint32_t kit = 0;
      for (int tile = 0; tile < ntiles; ++tile) {
        const int n0 = (int)(row0 + (int64_t)tile * kTileN) + (int)rank * (kTileN / 2);
        for (int mp = 0; mp < n_mp; ++mp) {
          const int q0 = mp * kPairM + (int)rank * kTileM;
          for (int kc = 0; kc < nk; ++kc, ++kit) {
            const int s = kit % kStages2;
            const uint32_t ph = (kit / kStages2) & 1;
            mbar_wait(&empty[s], ph ^ 1);
            uint8_t* sa = smem + s * kStage2Bytes;
            uint8_t* sb = sa + kA2Bytes;
            if (rank == 0) mbar_arrive_expect_tx(&full[s], 2 * kStage2Bytes);
            uint32_t fl = full_leader[0];
#pragma unroll
            for (int j = 1; j < kStages2; ++j) fl = (s == j) ? full_leader[j] : fl;
            tma_load_2d_pair(sa, &tm_q, kc * kTileK, q0, fl);
            tma_load_2d_pair(sb, &tm_bank, kc * kTileK, n0, fl);
            tma_load_2d_pair(sb + kBoxN * kTileK * 2, &tm_bank, kc * kTileK, n0 + kBoxN, fl);
          }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ===== MMA issuer (leader CTA only) =====
    if (lane == 0 && rank == 0) {
      const uint32_t idesc = make_idesc(kPairM, kTileN);
      uint32_t kit = 0, it = 0;
      for (int tile = 0; tile < ntiles; ++tile) {
        for (int mp = 0; mp < n_mp; ++mp, ++it) {
          const uint32_t acc = it & 1, aph = (it >> 1) & 1;
          mbar_wait(&tempty[acc], aph ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + acc * kTileN;
          for (int kc = 0; kc < nk; ++kc, ++kit) {
            const int s = kit % kStages2;
            const uint32_t ph = (kit / kStages2) & 1;
            mbar_wait(&full[s], ph);
            tc_fence_after();
            const uint32_t sa = smem_u32(smem + s * kStage2Bytes);
            const uint64_t adesc = make_smem_desc(sa);
            const uint64_t bdesc = make_smem_desc(sa + kA2Bytes);
#pragma unroll
            for (int k4 = 0; k4 < kTileK / 16; ++k4)
              tc_mma_pair(d_tmem, adesc + 2 * k4, bdesc + 2 * k4, idesc, (uint32_t)((kc | k4) != 0));
            tc_commit_pair(&empty[s]);
          }
          tc_commit_pair(&tfull[acc]);
        }
      }
    }
    __syncwarp();
  } else if (warp < 6) {
    // ===== epilogue (both CTAs): fused per-query top-KCAP =====
    const int quarter = warp & 3;
    const int tl = quarter * 32 + lane;
    const uint32_t tempty_leader[2] = {mapa_u32(smem_u32(&tempty[0]), 0), mapa_u32(smem_u32(&tempty[1]), 0)};
    Visit<KCAP> st;
    grid_dependency_wait();   // gthr was cleared by the preceding kernel
    uint32_t g_cur = 0;       // best published lower bound of this visit's query, fetched during the previous visit
    uint32_t it = 0;
    for (int tile = 0; tile < ntiles; ++tile) {
      const int n0 = (int)(row0 + (int64_t)tile * kTileN);
      const int c_end = (int)min((int64_t)kTileN, N - (int64_t)n0);   // rows >= N are TMA zero fill
      for (int mp = 0; mp < n_mp; ++mp, ++it) {
        const uint32_t acc = it & 1, aph = (it >> 1) & 1;
        const int r = mp * kPairM + (int)rank * kTileM + tl;
        const bool warp_active = (mp * kPairM + (int)rank * kTileM + quarter * 32) < B;   // warp-uniform
        const size_t pbase = ((size_t)cl * (size_t)Bpad + (size_t)r) * KCAP;
        float4* ps4 = reinterpret_cast<float4*>(part_sim + pbase);
        int4* pi4 = reinterpret_cast<int4*>(part_idx + pbase);
        const int r_nxt = ((mp + 1 == n_mp) ? 0 : mp + 1) * kPairM + (int)rank * kTileM + tl;
        const uint32_t g_nxt = (r_nxt < B) ? *reinterpret_cast<volatile uint32_t*>(gthr + r_nxt) : 0u;
        st.cnt = 0;
        st.loaded = false;
        st.thr = INFINITY;   // padding lanes never collect
        if (r < B) {
          float own = -INFINITY;   // K-th best of this (slab, query) list so far
          uint32_t gl = 0;         // pooled bound of this query (ordered; 0 = none)
          if (tile == 0) {
#pragma unroll
            for (int j = 0; j < KCAP; ++j) { st.v[j] = -INFINITY; st.ix[j] = -1; }
            st.loaded = true;
          } else {
            own = thr_s[mp * kTileM + tl];
            gl = *reinterpret_cast<volatile uint32_t*>(gl_s + mp * kTileM + tl);   // written by the refresher warp
          }
          // Admission threshold: above the list's own K-th best (strictly: an equal similarity met later has a
          // larger index), and not below what bounds the query's GLOBAL (k + slack)-th best from below: the pooled
          // bound, and the best K-th best any single slab has published (an EQUAL similarity may still belong to
          // the global best, hence the -1 in the ordered domain).
          uint32_t ge = g_cur > gl ? g_cur : gl;
          ge = ge ? ge - 1u : 0u;
          const uint32_t lo = f32_ordered(own);
          st.thr = f32_unordered(lo > ge ? lo : ge);
        }
        mbar_wait(&tfull[acc], aph);
        tc_fence_after();
        if (warp_active) {
          // the accumulator always holds 256 columns (columns >= c_end are similarities to zero-filled rows)
          const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + acc * kTileN;
          if constexpr (KCAP <= 16) {
            // TMEM reads (64 B/clk) bound the visit: the next 64 columns are in flight while these are folded
            uint32_t ra[32], rb[32], rc[32], rd[32];
            tmem_ld32(taddr, ra);
            tmem_ld32(taddr + 32, rb);
#pragma unroll 1
            for (int c0 = 0; c0 < kTileN; c0 += 128) {
              tmem_ld_wait();
              tmem_ld32(taddr + c0 + 64, rc);
              tmem_ld32(taddr + c0 + 96, rd);
              if (c0 < c_end) park_chunk<KCAP>(ra, c0, c_end, n0, st, ps4, pi4, cand, tl);
              if (c0 + 32 < c_end) park_chunk<KCAP>(rb, c0 + 32, c_end, n0, st, ps4, pi4, cand, tl);
              tmem_ld_wait();
              if (c0 + 128 < kTileN) {
                tmem_ld32(taddr + c0 + 128, ra);
                tmem_ld32(taddr + c0 + 160, rb);
              }
              if (c0 + 64 < c_end) park_chunk<KCAP>(rc, c0 + 64, c_end, n0, st, ps4, pi4, cand, tl);
              if (c0 + 96 < c_end) park_chunk<KCAP>(rd, c0 + 96, c_end, n0, st, ps4, pi4, cand, tl);
            }
          } else {
            for (int c0 = 0; c0 < c_end; c0 += 32) {
              uint32_t ra[32];
              tmem_ld32(taddr + c0, ra);
              tmem_ld_wait();
              park_chunk<KCAP>(ra, c0, c_end, n0, st, ps4, pi4, cand, tl);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(tempty_leader[acc]);   // accumulator released; now the insertions
        if (warp_active && __any_sync(0xffffffffu, st.cnt > 0)) drain<KCAP>(st, ps4, pi4, cand, tl, n0);
        if (st.loaded) {
#pragma unroll
          for (int j = 0; j < KCAP / 4; ++j) {
            ps4[j] = make_float4(st.v[4 * j], st.v[4 * j + 1], st.v[4 * j + 2], st.v[4 * j + 3]);
            pi4[j] = make_int4(st.ix[4 * j], st.ix[4 * j + 1], st.ix[4 * j + 2], st.ix[4 * j + 3]);
          }
          const float own = st.v[KCAP - 1];
          thr_s[mp * kTileM + tl] = own;
          // (a list shorter than k + slack proves nothing about the global (k + slack)-th best: only the pooled bound then)
          if (publish_own && own > -INFINITY) atomicMax(gthr + r, f32_ordered(own));
          const float pj = pub_j == 1 ? st.v[0] : (pub_j == 2 ? st.v[1] : (pub_j == 3 ? st.v[2] : st.v[3]));
          if (pj > -INFINITY) gthr[(size_t)Bpad * (1 + cl) + r] = f32_ordered(pj);
        }
        g_cur = g_nxt;
      }
    }
    __syncwarp();
    if (lane == 0) atomicAdd(epi_done, 1);
  } else {
    // ===== bound refresher (both CTAs) =====
    // Every slab publishes, per query, the pub_j-th best similarity it has met (gthr + Bpad * (1 + slab)).  The
    // G-th largest of those values over all slabs, G = pub_groups, has G * pub_j >= k + slack entries of the bank
    // at or above it, so it bounds the query's global (k + slack)-th best from below -- with ~74 slabs it is close
    // to the threshold a single stream over all rows seen so far would have.  This warp recomputes it for the
    // CTA's queries round and round until the epilogue is done; the epilogue reads it from shared memory.
    grid_dependency_wait();
    const volatile int* done = epi_done;
    while (*done < 4) {
      for (int mp = 0; mp < n_mp && *done < 4; ++mp) {
        for (int q4 = (warp - 6) * 2; q4 < (warp - 6) * 2 + 2; ++q4) {   // each refresher warp serves 64 of the 128 queries
          const int tq = q4 * 32 + lane;
          const int r = mp * kPairM + (int)rank * kTileM + tq;
          if (mp * kPairM + (int)rank * kTileM + q4 * 32 >= B) break;   // warp-uniform
          uint32_t top[16];   // the G largest published values, descending (G <= 16)
#pragma unroll
          for (int j = 0; j < 16; ++j) top[j] = 0u;
          if (r < B) {
            const volatile uint32_t* pub = gthr + (size_t)Bpad + r;
#pragma unroll 2
            for (int c = 0; c < ncl; ++c) {
              const uint32_t x = pub[(size_t)c * Bpad];
              if (x > top[15]) {
#pragma unroll
                for (int j = 15; j >= 1; --j) {
                  const bool up = x > top[j - 1];
                  top[j] = up ? top[j - 1] : (x > top[j] ? x : top[j]);
                }
                top[0] = x > top[0] ? x : top[0];
              }
            }
            uint32_t tau = top[0];
#pragma unroll
            for (int j = 1; j < 16; ++j) tau = (j < pub_groups) ? top[j] : tau;
            if (pub_groups > 16) tau = 0u;
            const uint32_t old = gl_s[mp * kTileM + tq];
            if (tau > old) gl_s[mp * kTileM + tq] = tau;
          }
        }
      }
    }
  }

  tc_fence_before();
  cluster_sync_all();   // the leader's MMAs read the peer's shared memory and write its TMEM: leave together
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

}  // namespace


cudaError_t scan_tc2_prepare() {
  cudaError_t e;
  e = cudaFuncSetAttribute(scan_tc2_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem2Bytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(scan_tc2_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem2Bytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(scan_tc2_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem2Bytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(scan_tc2_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem2Bytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(scan_tc2_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem2Bytes);
}

int scan_tc2_clusters(int64_t N, int max_grid) {
  const int64_t tiles = (N + kTileN - 1) / kTileN;
  const int64_t ncl = max_grid / 2;
  return (int)(tiles < ncl ? tiles : ncl);
}

cudaError_t launch_scan_tc2(const CUtensorMap* tm_q, const CUtensorMap* tm_bank, int64_t N, int d, int B, int Bpad,
                            int kcap, int kc, int max_grid, float* part_sim, int32_t* part_idx, uint32_t* gthr,
                            int* clusters_out, cudaStream_t s) {
  const int ncl = scan_tc2_clusters(N, max_grid);
  if (clusters_out) *clusters_out = ncl;
  const int pub_j = (kc + 15) / 16, pub_groups = (kc + pub_j - 1) / pub_j;   // pub_groups * pub_j >= kc
  cudaError_t e = cudaSuccess;
#define RB_SCAN2_LAUNCH(KC)                                                                                       \
  e = launch_chained(scan_tc2_kernel<KC>, dim3(2 * ncl), dim3(kThreads2), kSmem2Bytes, s, *tm_q, *tm_bank, N, d, B, Bpad, \
                     part_sim, part_idx, gthr, pub_j, pub_groups, kcap >= kc ? 1 : 0)
  switch (kcap) {
    case 4: RB_SCAN2_LAUNCH(4); break;
    case 8: RB_SCAN2_LAUNCH(8); break;
    case 16: RB_SCAN2_LAUNCH(16); break;
    case 32: RB_SCAN2_LAUNCH(32); break;
    default: RB_SCAN2_LAUNCH(64); break;
  }
#undef RB_SCAN2_LAUNCH
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rb
