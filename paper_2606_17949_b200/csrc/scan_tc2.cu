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
// the list's last similarity (the admission threshold) and touches the list itself only when a candidate
// beats it -- rare after the first tiles.
#include "rb_internal.cuh"
#include "tc_scan.cuh"

namespace rb {
namespace {

constexpr int kStages2 = 6;
constexpr int kA2Bytes = kTileM * kTileK * 2;            // 16 KB: this CTA's 128 queries x 64 bf16
constexpr int kB2Bytes = (kTileN / 2) * kTileK * 2;      // 16 KB: this CTA's 128 of the tile's 256 bank rows
constexpr int kStage2Bytes = kA2Bytes + kB2Bytes;        // 32 KB
constexpr int kThreads2 = 192;
constexpr int kSmem2Bytes = kStages2 * kStage2Bytes + kCandSlots * kTileM * 8 + 256 + 1024;
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
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
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

// One tcgen05.ld chunk folded into the thread's list, the list itself fetched from global memory only when this
// thread has a candidate above its threshold (tc_scan.cuh: fold_chunk is the register-resident variant).
template <int K>
__device__ __forceinline__ void fold_chunk_lazy(const uint32_t (&regs)[32], int c0, int c_end, int n0, float (&v)[K],
                                                int32_t (&ix)[K], float& thr, bool& loaded, const float4* ps4,
                                                const int4* pi4, uint2* cand, int tl) {
  const bool full = c0 + 32 <= c_end;   // warp-uniform
  float m0 = -INFINITY, m1 = -INFINITY, m2 = -INFINITY, m3 = -INFINITY;
#pragma unroll
  for (int j = 0; j < 32; j += 4) {
    m0 = fmaxf(m0, (full || c0 + j + 0 < c_end) ? __uint_as_float(regs[j + 0]) : -INFINITY);
    m1 = fmaxf(m1, (full || c0 + j + 1 < c_end) ? __uint_as_float(regs[j + 1]) : -INFINITY);
    m2 = fmaxf(m2, (full || c0 + j + 2 < c_end) ? __uint_as_float(regs[j + 2]) : -INFINITY);
    m3 = fmaxf(m3, (full || c0 + j + 3 < c_end) ? __uint_as_float(regs[j + 3]) : -INFINITY);
  }
  const float m = fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
  if (!__any_sync(0xffffffffu, m > thr)) return;
  int cnt = 0;
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    const float s = __uint_as_float(regs[j]);
    if ((full || c0 + j < c_end) && s > thr) {
      cand[cnt * kTileM + tl] = make_uint2(regs[j], (uint32_t)(c0 + j));
      ++cnt;
    }
  }
  if (cnt > 0 && !loaded) {
#pragma unroll
    for (int j = 0; j < K / 4; ++j) {
      const float4 a = ps4[j];
      const int4 b = pi4[j];
      v[4 * j] = a.x; v[4 * j + 1] = a.y; v[4 * j + 2] = a.z; v[4 * j + 3] = a.w;
      ix[4 * j] = b.x; ix[4 * j + 1] = b.y; ix[4 * j + 2] = b.z; ix[4 * j + 3] = b.w;
    }
    loaded = true;
  }
  uint2 nxt = cand[tl];
  for (int p = 0; __any_sync(0xffffffffu, p < cnt); ++p) {
    const uint2 cur = nxt;
    nxt = cand[min(p + 1, kCandSlots - 1) * kTileM + tl];
    const float s = __uint_as_float(cur.x);
    if (p < cnt && s > thr) {
      list_insert<K>(v, ix, s, n0 + (int)cur.y);
      thr = v[K - 1];
    }
  }
}

template <int KCAP>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads2, 1)
scan_tc2_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_bank, int64_t N, int d,
                int B, int Bpad, float* part_sim, int32_t* part_idx) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint2* cand = (uint2*)(smem + kStages2 * kStage2Bytes);
  uint64_t* bars = (uint64_t*)(cand + kCandSlots * kTileM);
  uint64_t* full = bars;                   // [kStages2] leader's: both CTAs' TMA bytes landed
  uint64_t* empty = bars + kStages2;       // [kStages2] own: the MMAs that read the slot retired
  uint64_t* tfull = bars + 2 * kStages2;   // [2] own: accumulator complete
  uint64_t* tempty = tfull + 2;            // [2] leader's: accumulator drained by the 8 epilogue warps of the pair
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

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
  } else {
    // ===== epilogue (both CTAs): fused per-query top-KCAP =====
    const int quarter = warp & 3;
    const int tl = quarter * 32 + lane;
    const uint32_t tempty_leader[2] = {mapa_u32(smem_u32(&tempty[0]), 0), mapa_u32(smem_u32(&tempty[1]), 0)};
    float v[KCAP];
    int32_t ix[KCAP];
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
        bool loaded = false;
        float thr = INFINITY;   // padding lanes never collect
        if (warp_active && r < B) {
          if (tile == 0) {
#pragma unroll
            for (int j = 0; j < KCAP; ++j) { v[j] = -INFINITY; ix[j] = -1; }
            loaded = true;
            thr = -INFINITY;
          } else {
            thr = *reinterpret_cast<volatile float*>(part_sim + pbase + KCAP - 1);
          }
        }
        mbar_wait(&tfull[acc], aph);
        tc_fence_after();
        if (warp_active) {
          const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + acc * kTileN;
          if constexpr (KCAP <= 16) {
            for (int c0 = 0; c0 < c_end; c0 += 64) {
              uint32_t ra[32], rb[32];
              const bool two = c0 + 32 < c_end;
              tmem_ld32(taddr + c0, ra);
              if (two) tmem_ld32(taddr + c0 + 32, rb);
              tmem_ld_wait();
              fold_chunk_lazy<KCAP>(ra, c0, c_end, n0, v, ix, thr, loaded, ps4, pi4, cand, tl);
              if (two) fold_chunk_lazy<KCAP>(rb, c0 + 32, c_end, n0, v, ix, thr, loaded, ps4, pi4, cand, tl);
            }
          } else {
            for (int c0 = 0; c0 < c_end; c0 += 32) {
              uint32_t ra[32];
              tmem_ld32(taddr + c0, ra);
              tmem_ld_wait();
              fold_chunk_lazy<KCAP>(ra, c0, c_end, n0, v, ix, thr, loaded, ps4, pi4, cand, tl);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(tempty_leader[acc]);
        if (loaded) {
#pragma unroll
          for (int j = 0; j < KCAP / 4; ++j) {
            ps4[j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
            pi4[j] = make_int4(ix[4 * j], ix[4 * j + 1], ix[4 * j + 2], ix[4 * j + 3]);
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
                            int kcap, int max_grid, float* part_sim, int32_t* part_idx, int* clusters_out, cudaStream_t s) {
  const int ncl = scan_tc2_clusters(N, max_grid);
  if (clusters_out) *clusters_out = ncl;
  cudaError_t e = cudaSuccess;
#define RB_SCAN2_LAUNCH(KC)                                                                                       \
  e = launch_chained(scan_tc2_kernel<KC>, dim3(2 * ncl), dim3(kThreads2), kSmem2Bytes, s, *tm_q, *tm_bank, N, d, B, Bpad, \
                     part_sim, part_idx)
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
