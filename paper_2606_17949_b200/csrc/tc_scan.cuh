// tc_scan.cuh -- what the two tensor-core scan kernels (scan_tc.cu: one CTA per SM, scan_tc2.cu: CTA pairs) share:
// PTX wrappers for mbarrier / TMA / tcgen05, the shared-memory and instruction descriptors, and the fused
// per-thread top-K fold of one tcgen05.ld chunk.  Product code; included by those two files only.
#pragma once
#include "rb_internal.cuh"

namespace rb {
namespace {

constexpr int kCandSlots = 32;                     // one tcgen05.ld chunk can yield at most 32 survivors

// Order-preserving map float -> uint32 (larger float = larger uint) and back.
__device__ __forceinline__ uint32_t f32_ordered(float f) {
  const uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float f32_unordered(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}

// ---- PTX wrappers (mbarrier wrappers: rb_internal.cuh) ----------------------------------------------------
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, bf16 x bf16 -> fp32, one 128 x N x 16 step.
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accum)
      : "memory");
}
// 32 lanes x 32 consecutive fp32 columns: thread t of the warp receives lane (base lane + t).
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor: K-major operand, 128-byte swizzle, rows of 128 bytes, 8-row groups 1024 B apart.
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
  uint64_t desc = 0;
  desc |= (uint64_t)((saddr & 0x3FFFF) >> 4);        // start address
  desc |= (uint64_t)0 << 16;                          // leading-dimension byte offset: unused for swizzled K-major
  desc |= (uint64_t)(1024 >> 4) << 32;                // stride-dimension byte offset
  desc |= (uint64_t)1 << 46;                          // descriptor version (sm_100)
  desc |= (uint64_t)2 << 61;                          // SWIZZLE_128B
  return desc;
}
// Instruction descriptor, kind::f16: D fp32, A = B = bf16, both K-major, M x N.
__device__ __forceinline__ uint32_t make_idesc(int m, int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}

// Sorted insertion into a register-resident list (similarity descending; an equal similarity goes after the
// entries already present, which have smaller bank indices because rows are scanned in ascending order).
template <int K>
__device__ __forceinline__ void list_insert(float (&v)[K], int32_t (&ix)[K], float s, int32_t id) {
#pragma unroll
  for (int j = K - 1; j >= 1; --j) {
    const bool up = s > v[j - 1];
    const bool here = (!up) && (s > v[j]);
    const float nv = up ? v[j - 1] : (here ? s : v[j]);
    const int32_t ni = up ? ix[j - 1] : (here ? id : ix[j]);
    v[j] = nv;
    ix[j] = ni;
  }
  const bool top = s > v[0];
  v[0] = top ? s : v[0];
  ix[0] = top ? id : ix[0];
}

// One tcgen05.ld chunk (32 similarities of this thread's query against bank rows n0+c0 ..) folded into the
// thread's sorted list.  Steady state: no lane of the warp holds a similarity above its threshold and the chunk
// costs one max tree and one vote.  Otherwise the survivors (rare after warm-up) are parked in shared memory
// and inserted in warp lock-step: every lane inserts its p-th survivor in the same iteration, so there is one
// copy of the insertion code (the epilogue runs on few warps; its code must stay small).
template <int K>
__device__ __forceinline__ void fold_chunk(const uint32_t (&regs)[32], int c0, int c_end, int n0, float (&v)[K],
                                           int32_t (&ix)[K], float& thr, uint2* cand, int tl) {
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
  uint2 nxt = cand[tl];
  for (int p = 0; __any_sync(0xffffffffu, p < cnt); ++p) {
    const uint2 cur = nxt;
    nxt = cand[min(p + 1, kCandSlots - 1) * kTileM + tl];   // next survivor's slot is read while this one is inserted
    const float s = __uint_as_float(cur.x);
    if (p < cnt && s > thr) {
      list_insert<K>(v, ix, s, n0 + (int)cur.y);
      thr = v[K - 1];
    }
  }
}

}  // namespace
}  // namespace rb
