// scan_tc.cu -- step a1 for bf16 storage: similarity scan of the reference bank on the 5th-gen tensor cores
// with a fused per-query top-KCAP epilogue.  The B x N similarity matrix exists only in TMEM.
//
// Definition ("queries a ... KNN index (k=10) over the 14,919-prompt training split"; DESIGN.md
// readings 1, 3, 4): s[r,n] = <q~_r, e~_n> over the bf16-rounded vectors; keep, per query, the best entries in
// the order (s descending, n ascending).  Here each CTA keeps the best KCAP of its own slab of bank rows; the
// cross-CTA merge and the exact re-rank are finish_kernel (estimate.cu).
//
// Shape of the kernel (one persistent CTA per SM, 6 warps):
//   warp 0   TMA producer: cp.async.bulk.tensor tiles of the bank (64 rows x 64 bf16, 128B swizzle) and of the
//            staged queries (128 x 64) into a 4-stage shared-memory ring, mbarrier complete_tx.
//   warp 1   allocates TMEM (512 columns = two 128x256 fp32 accumulators) and issues tcgen05.mma
//            (M=128 queries x N<=256 bank rows x K=16) from one lane; tcgen05.commit releases ring slots and
//            publishes finished accumulators.
//   warps 2-5  epilogue: thread t owns TMEM lane t = query t of the m-tile; tcgen05.ld 32 columns at a time,
//            compare against the thread's current KCAP-th best similarity, append the rare survivors to a
//            shared-memory buffer, then insert them into a sorted register list in warp lock-step.
// Bank rows are split over CTAs in groups of 16 rows (the remainder of a slab's last tile is loaded through a second
// tensor map with 16-row boxes); a CTA walks its slab in tiles of 256 rows and, for
// B > 128, revisits each tile once per 128-query m-tile (bank tile then comes from L2), carrying the lists
// through global memory between visits.  For B <= 64 the queries are replicated over the lane quarters so that
// all four epilogue warps share the columns of a tile (the epilogue of a short slab is latency-bound).
// A CTA's lists leave as 32-byte records of the finishing kernel's 64-bit keys (order-preserving image of the similarity,
// ~index), query-major: the finishing CTA of a query reads them as one contiguous stream.
#include "rb_internal.cuh"
#include "tc_scan.cuh"

namespace rb {
namespace {


constexpr int kStages = 4;
constexpr int kABytes = kTileM * kTileK * 2;       // 16 KB: 128 queries x 64 bf16
constexpr int kBoxBytes = kBoxN * kTileK * 2;      //  8 KB: 64 bank rows x 64 bf16
constexpr int kBBytes = kTileN * kTileK * 2;       // 32 KB
constexpr int kStageBytes = kABytes + kBBytes;     // 48 KB
constexpr int kThreads = 192;
constexpr int kSmemBytes = kStages * kStageBytes + kCandSlots * kTileM * 8 + 256 + 1024;

template <int KCAP>
__global__ void __launch_bounds__(kThreads, 1)
scan_tc_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_bank,
               const __grid_constant__ CUtensorMap tm_bank16, int64_t N, int d, int B, int Bpad, int rep, float* __restrict__ part_sim, int32_t* __restrict__ part_idx,
               unsigned long long* __restrict__ dev_clock) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 128B swizzle wants 1024 B alignment
  uint2* cand = (uint2*)(smem + kStages * kStageBytes);   // [kCandSlots][128]: (similarity bits, column)
  uint64_t* bars = (uint64_t*)(cand + kCandSlots * kTileM);
  uint64_t* full = bars;                  // [kStages] TMA bytes landed
  uint64_t* empty = bars + kStages;       // [kStages] MMAs that read the slot retired
  uint64_t* tfull = bars + 2 * kStages;   // [2] accumulator complete
  uint64_t* tempty = tfull + 2;           // [2] accumulator drained by the epilogue
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_mt = Bpad / kTileM;
  const int nk = (d + kTileK - 1) / kTileK;
  // This CTA's rows: the bank is split in groups of kRowUnit = 16 rows (what the MMA's N and the 16-row boxes of tm_bank16
  // resolve), so the CTAs' shares differ by at most 16 rows -- with 64-row units C2 gave 83 CTAs 11 units and 65 CTAs 10,
  // and the last 10 % of the stream ran on 56 % of the SMs (CTA ends spread over 3.7 us of 24).
  const int64_t units = (N + kRowUnit - 1) / kRowUnit;
  const int64_t u0 = units * blockIdx.x / gridDim.x;
  const int64_t u1 = units * (blockIdx.x + 1) / gridDim.x;
  const int nrows = (int)(u1 - u0) * kRowUnit;
  const int64_t row0 = u0 * kRowUnit;
  const int ntiles = (nrows + kTileN - 1) / kTileN;

  launch_dependents();
  if (dev_clock != nullptr && threadIdx.x == 0) {   // stage-timing mode: earliest CTA start on the device's own clock
    unsigned long long t0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    atomicMin(dev_clock, t0);
  }
  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_q) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_bank) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_bank16) : "memory");
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&tfull[a], 1);
      mbar_init(&tempty[a], 4);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      grid_dependency_wait();   // the staged queries come from the preceding kernel (it ends about when this
                                // kernel's prologue does: issuing bank boxes ahead of the wait only delayed the
                                // first query tile behind them -- measured, reverted)
      uint32_t kit = 0;
      for (int tile = 0; tile < ntiles; ++tile) {
        const int n0 = (int)(row0 + (int64_t)tile * kTileN);
        const int trows = min(kTileN, nrows - tile * kTileN);   // a multiple of 16
        const int nun = trows / kBoxN, n16 = (trows % kBoxN) / kRowUnit;
        for (int mt = 0; mt < n_mt; ++mt) {
          for (int kc = 0; kc < nk; ++kc, ++kit) {
            const int s = kit % kStages;
            const uint32_t ph = (kit / kStages) & 1;
            mbar_wait(&empty[s], ph ^ 1);
            uint8_t* sa = smem + s * kStageBytes;
            uint8_t* sb = sa + kABytes;
            mbar_arrive_expect_tx(&full[s], kABytes + trows * kTileK * 2);
            tma_load_2d(sa, &tm_q, kc * kTileK, mt * kTileM, &full[s]);
            for (int u = 0; u < nun; ++u) tma_load_2d(sb + u * kBoxBytes, &tm_bank, kc * kTileK, n0 + u * kBoxN, &full[s]);
            // (the rest of a last tile: 16-row boxes, laid out like a quarter of a 64-row box -- the swizzle repeats every 8 rows)
            for (int u = 0; u < n16; ++u)
              tma_load_2d(sb + nun * kBoxBytes + u * (kBoxBytes / 4), &tm_bank16, kc * kTileK, n0 + nun * kBoxN + u * kRowUnit, &full[s]);
          }
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0) {
      uint32_t kit = 0, it = 0;
      for (int tile = 0; tile < ntiles; ++tile) {
        const int trows = min(kTileN, nrows - tile * kTileN);
        const uint32_t idesc = make_idesc(kTileM, trows);
        for (int mt = 0; mt < n_mt; ++mt, ++it) {
          const uint32_t acc = it & 1, aph = (it >> 1) & 1;
          mbar_wait(&tempty[acc], aph ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + acc * kTileN;
          for (int kc = 0; kc < nk; ++kc, ++kit) {
            const int s = kit % kStages;
            const uint32_t ph = (kit / kStages) & 1;
            mbar_wait(&full[s], ph);
            tc_fence_after();
            const uint32_t sa = smem_u32(smem + s * kStageBytes);
            const uint64_t adesc = make_smem_desc(sa);
            const uint64_t bdesc = make_smem_desc(sa + kABytes);
#pragma unroll
            for (int k4 = 0; k4 < kTileK / 16; ++k4) {
              // +32 bytes along K inside the 128-byte swizzle row = +2 in the encoded start address
              tc_mma(d_tmem, adesc + 2 * k4, bdesc + 2 * k4, idesc, (uint32_t)((kc | k4) != 0));
            }
            tc_commit(&empty[s]);
          }
          tc_commit(&tfull[acc]);
        }
      }
    }
    __syncwarp();
  } else {
    // ===== epilogue: fused per-query top-KCAP =====
    // rep = 4 (B <= 32) / 2 (B <= 64): the staged queries are replicated over the TMEM lane quarters, so each
    // quarter's warp sees every query and folds its own share of the tile's columns into its own list
    // (list index = CTA * rep + replica).  rep = 1: one query per TMEM lane, all columns.
    const int quarter = warp & 3;              // TMEM lane quarter this warp may read
    const int tl = quarter * 32 + lane;        // TMEM lane inside the m-tile
    const int group = kTileM / rep;            // lanes per replica
    const int replica = tl / group;
    float v[KCAP];
    int32_t ix[KCAP];
    uint32_t it = 0;
    for (int tile = 0; tile < ntiles; ++tile) {
      const int n0 = (int)(row0 + (int64_t)tile * kTileN);
      const int ncols = min(kTileN, nrows - tile * kTileN);
      const int nvalid = (int)min((int64_t)ncols, N - (int64_t)n0);   // rows >= N are TMA zero fill
      // the replicas share the tile's columns in runs of 32 (one TMEM load): a short last tile is spread over all of them
      const int cpr = ((ncols + rep - 1) / rep + 31) & ~31;
      const int col_lo = replica * cpr;
      const int c_end = min(col_lo + cpr, nvalid);
      for (int mt = 0; mt < n_mt; ++mt, ++it) {
        const uint32_t acc = it & 1, aph = (it >> 1) & 1;
        const int r = mt * kTileM + (tl - replica * group);
        const bool warp_active = (mt * kTileM + (quarter * 32) % group) < B;   // warp-uniform
        // query-major 32-byte records [similarities of a quad | their indices]: the finishing CTA of a query reads its
        // lists as one contiguous stream of whole sectors (a half-written sector would cost it a DRAM fill)
        const size_t pbase = ((size_t)r * ((size_t)gridDim.x * rep) + ((size_t)blockIdx.x * rep + replica)) * (KCAP / 4) * 2;
        uint4* prec = reinterpret_cast<uint4*>(part_sim) + pbase;
        if (warp_active) {
          if (tile == 0) {
#pragma unroll
            for (int j = 0; j < KCAP; ++j) { v[j] = -INFINITY; ix[j] = -1; }
          } else if (n_mt > 1) {
#pragma unroll
            for (int j = 0; j < KCAP / 4; ++j) {   // records hold keys (see the store below): decode them
              const uint4 ua = prec[2 * j], ub = prec[2 * j + 1];
              const uint32_t lo[4] = {ua.x, ua.z, ub.x, ub.z}, hi[4] = {ua.y, ua.w, ub.y, ub.w};
#pragma unroll
              for (int h = 0; h < 4; ++h) {
                const bool real = (lo[h] | hi[h]) != 0u;
                v[4 * j + h] = real ? f32_unordered(hi[h]) : -INFINITY;
                ix[4 * j + h] = real ? (int32_t)(0xffffffffu - lo[h]) : -1;
              }
            }
          }
        }
        mbar_wait(&tfull[acc], aph);
        tc_fence_after();
        if (warp_active) {
          float thr = (r < B) ? v[KCAP - 1] : INFINITY;   // padding lanes never collect
          const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + acc * kTileN;
          if constexpr (KCAP <= 16) {   // two loads in flight per wait; longer lists need the registers
            for (int c0 = col_lo; c0 < c_end; c0 += 64) {
              uint32_t ra[32], rb[32];
              const bool two = c0 + 32 < c_end;   // warp-uniform; the accumulator holds a multiple of 64 columns
              tmem_ld32(taddr + c0, ra);
              if (two) tmem_ld32(taddr + c0 + 32, rb);
              tmem_ld_wait();
              fold_chunk<KCAP>(ra, c0, c_end, n0, v, ix, thr, cand, tl);
              if (two) fold_chunk<KCAP>(rb, c0 + 32, c_end, n0, v, ix, thr, cand, tl);
            }
          } else {
            for (int c0 = col_lo; c0 < c_end; c0 += 32) {
              uint32_t ra[32];
              tmem_ld32(taddr + c0, ra);
              tmem_ld_wait();
              fold_chunk<KCAP>(ra, c0, c_end, n0, v, ix, thr, cand, tl);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty[acc]);
        if (warp_active && r < B && (n_mt > 1 || tile == ntiles - 1)) {
#pragma unroll
          for (int j = 0; j < KCAP / 4; ++j) {
            // A record = the finishing kernel's 64-bit keys of a quad of entries, ready made: high word = the similarity's
            // order-preserving integer image, low word = ~index (larger key = better; 0 = empty slot).
            // One 256-bit store per record: the whole 32-byte sector in one transaction (two 16-byte stores would each be
            // a partial-sector write that L2 has to complete from DRAM)
            uint32_t kw[8];
#pragma unroll
            for (int h = 0; h < 4; ++h) {
              const bool real = ix[4 * j + h] >= 0;
              kw[2 * h] = real ? 0xffffffffu - (uint32_t)ix[4 * j + h] : 0u;
              kw[2 * h + 1] = real ? f32_ordered(v[4 * j + h]) : 0u;
            }
            asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(prec + 2 * j), "r"(kw[0]), "r"(kw[1]),
                         "r"(kw[2]), "r"(kw[3]), "r"(kw[4]), "r"(kw[5]), "r"(kw[6]), "r"(kw[7])
                         : "memory");
          }
        }
      }
    }
  }

  if (dev_clock != nullptr && warp >= 2 && lane == 0) {   // ... and latest CTA end: an epilogue warp, behind its last store
    // (a stamp taken by another warp behind the closing barrier reads the timer when the BAR.SYNC.DEFER_BLOCKING is
    // issued, not when it completes: it came out 2 us before the epilogue's own end)
    unsigned long long t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)::"memory");
    atomicMax(dev_clock + 1, t1);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

}  // namespace


size_t scan_tc_smem_bytes() { return kSmemBytes; }

cudaError_t scan_tc_prepare() {
  cudaError_t e;
  e = cudaFuncSetAttribute(scan_tc_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(scan_tc_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(scan_tc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(scan_tc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(scan_tc_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
}

int scan_tc_replicas(int B, int kcap, int max_grid) {
  int rep = B <= 32 ? 4 : (B <= 64 ? 2 : 1);
  while (rep > 1 && (size_t)max_grid * rep * kcap * 8 > (size_t)160 * 1024) rep >>= 1;
  return rep;
}

cudaError_t launch_scan_tc(const CUtensorMap* tm_q, const CUtensorMap* tm_bank, const CUtensorMap* tm_bank16, int64_t N, int d, int B, int Bpad,
                           int kcap, int max_grid, float* part_sim, int32_t* part_idx, int* grid_out,
                           unsigned long long* dev_clock, cudaStream_t s) {
  const int64_t units = (N + kBoxN - 1) / kBoxN;
  const int grid = (int)(units < max_grid ? units : max_grid);
  const int rep = scan_tc_replicas(B, kcap, max_grid);
  if (grid_out) *grid_out = grid;
  cudaError_t e = cudaSuccess;
#define RB_SCAN_LAUNCH(KC)                                                                                          \
  e = launch_chained(scan_tc_kernel<KC>, dim3(grid), dim3(kThreads), kSmemBytes, s, *tm_q, *tm_bank, *tm_bank16, N, d, B, Bpad, rep, \
                     part_sim, part_idx, dev_clock)
  switch (kcap) {
    case 4: RB_SCAN_LAUNCH(4); break;
    case 8: RB_SCAN_LAUNCH(8); break;
    case 16: RB_SCAN_LAUNCH(16); break;
    case 32: RB_SCAN_LAUNCH(32); break;
    default: RB_SCAN_LAUNCH(64); break;
  }
#undef RB_SCAN_LAUNCH
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace rb
