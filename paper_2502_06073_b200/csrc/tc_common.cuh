// tc_common.cuh — inline-PTX wrappers shared by the tcgen05 GEMM kernels (gemm_tc.cu, gemm_f16s.cu): mbarriers, bulk copies,
// UMMA shared-memory descriptors, tcgen05.mma / commit / ld / st, and the per-warp transposition tiles that turn
// row-per-lane register tiles into full-sector global accesses.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace allegro {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ float tf32_rna(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

__device__ __forceinline__ float tf32_trunc(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

// K-major, no swizzle: start address, LBO (k direction) and SBO (row-group direction) in 16-byte units; version 1 (sm_100)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity), "r"(2000u)   // suspend-time hint (ns): fewer polls, the kernels are issue-bound
        : "memory");
  }
}

__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate));
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

__device__ __forceinline__ void tmem_st4(uint32_t taddr, float4 x) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(__float_as_uint(x.x)),
               "r"(__float_as_uint(x.y)), "r"(__float_as_uint(x.z)), "r"(__float_as_uint(x.w))
               : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float* v) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}

// A warp owns 32 rows; each thread computes 16 consecutive columns of its own row.  Global traffic goes through a
// per-warp shared-memory tile so that one instruction touches 8 rows x 64 contiguous bytes (full sectors) instead of
// 32 rows x 16 bytes.  The tile is [32][16] floats with the 16-byte chunk index XOR-swizzled by (row >> 1) & 3: the
// row-per-lane side (8 lanes = 8 rows, one chunk each) and the transposed side (8 lanes = 2 rows x 4 chunks) are both free of
// bank conflicts (a padded 20-float row is not: rows r and r+1 of the transposed side overlap by four banks).
constexpr int WT_LD = 16;
__device__ __forceinline__ int wt_off(int r, int chunk) { return r * WT_LD + 4 * (chunk ^ ((r >> 1) & 3)); }
__device__ __forceinline__ void warp_tile_store(float* tile, const float4 (&o)[4], int lane, float* C, int ld, int64_t rbase, int64_t M,
                                                int col0, int N) {
#pragma unroll
  for (int j = 0; j < 4; ++j) *reinterpret_cast<float4*>(tile + wt_off(lane, j)) = o[j];
  __syncwarp();
  const int cq = (lane & 3) * 4;
  float4 t[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) t[i] = *reinterpret_cast<const float4*>(tile + wt_off(i * 8 + (lane >> 2), lane & 3));
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = i * 8 + (lane >> 2);
    if (rbase + r < M && col0 + cq < N) *reinterpret_cast<float4*>(C + (rbase + r) * ld + col0 + cq) = t[i];
  }
  __syncwarp();
}
// Asynchronous load side: cp.async writes the transposed side of a tile directly (no registers, zero fill outside the valid
// rows / columns); after cp.async.wait_group + __syncwarp the owner lanes read their rows with warp_tile_read.
__device__ __forceinline__ void warp_tile_prefetch(float* tile, int lane, const float* A, int ld, int64_t rbase, int64_t M, int col0, int N) {
  const int cq = (lane & 3) * 4;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = i * 8 + (lane >> 2);
    const bool ok = rbase + r < M && col0 + cq < N;
    const float* src = ok ? A + (rbase + r) * ld + col0 + cq : A;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(tile + wt_off(r, lane & 3))), "l"(src), "r"(ok ? 16u : 0u) : "memory");
  }
}
__device__ __forceinline__ void warp_tile_read(const float* tile, float4 (&x)[4], int lane) {
#pragma unroll
  for (int j = 0; j < 4; ++j) x[j] = *reinterpret_cast<const float4*>(tile + wt_off(lane, j));
}
// load side in two steps, so that the global loads of several row segments can be in flight before the first transposition
__device__ __forceinline__ void warp_tile_ldg(float4 (&t)[4], int lane, const float* A, int ld, int64_t rbase, int64_t M, int col0, int N) {
  const int cq = (lane & 3) * 4;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = i * 8 + (lane >> 2);
    t[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (rbase + r < M && col0 + cq < N) t[i] = *reinterpret_cast<const float4*>(A + (rbase + r) * ld + col0 + cq);
  }
}
__device__ __forceinline__ void warp_tile_xpose(float* tile, const float4 (&t)[4], float4 (&x)[4], int lane) {
#pragma unroll
  for (int i = 0; i < 4; ++i) *reinterpret_cast<float4*>(tile + wt_off(i * 8 + (lane >> 2), lane & 3)) = t[i];
  __syncwarp();
#pragma unroll
  for (int j = 0; j < 4; ++j) x[j] = *reinterpret_cast<const float4*>(tile + wt_off(lane, j));
  __syncwarp();
}

}  // namespace allegro
