// gemm_f16s.cu — the wide edge-by-width GEMMs (latent / two-body MLPs, W_init / W_env, channel mixing and their transposes;
// PAPER.md:93, Table 1) on tcgen05 with a split-fp16 operand format, for the networks whose widths exceed the chained kernel
// of gemm_tc.cu (BASELINE.json configs 2 and 3).  Same contract as k_gemm (gemm.cuh):  C = epi( pro(A) B ).
//
// Precision ("only in a precision that stays inside the stated tolerance", north_star).  The product is formed from three
// kind::f16 passes accumulated in fp32 in ONE TMEM accumulator (an error-corrected split in the manner of Ootomo & Yokota 2022,
// restated for the operand formats of this instruction, which takes fp16 x fp16 or bf16 x bf16 — a mixed pair traps):
//   activations  x = a_hi + a_lo,  a_hi = fp16(x) (11 significant bits),  a_lo = bf16(x - a_hi) (8 more bits; bf16 has the exponent
//                range of fp32, so a_lo needs no scaling whatever the magnitude of x: |x - a_hi - a_lo| <= 2^-21 |x|)
//   weights      w' = 2^s w with s per matrix such that max |w'| is in [2^13, 2^14) (exact; 2^-s is applied to the accumulator in the
//                epilogue);  b_hi = fp16(w'),  b_lo = fp16(w' - b_hi)  (normal numbers thanks to the scaling: 22 bits),  b_b = bf16(w')
//   A W ~= a_hi b_hi + a_hi b_lo  (fp16 x fp16)  +  a_lo b_b  (bf16 x bf16)
// dropped: a_lo (w' - b_b) <= 2^-12 2^-9 and the 2^-21 above, i.e. ~1e-6 per product at worst, ~3e-7 RMS.  It runs at twice the
// tensor-pipe rate of the 3 x TF32 split of gemm_tc.cu.  One accumulator (256 of the 512 TMEM columns per 128 x 256 tile) is what
// lets the accumulators be double-buffered: the epilogue of a tile runs under the k loop of the next.  (Round 2 first used
// lo = fp16((x - hi) 2048) on both sides, 2 x 11 bits, which needs a second accumulator for the scaled terms and so fills TMEM:
// epilogue and k loop were serial.)  |x| >= 65520 overflows fp16 (the force call then ends with ALLEGRO_ERR_NONFINITE);
// DESIGN.md R4 has the measured error table for 1, 2 and 3 passes.
//
// One persistent CTA per SM (21 warps), tiles of 128 rows x up to 256 columns, K in stages of 32 (3 stages of 64 KB):
//   * 2 warps issue the TMA loads of the raw fp32 A stage (128 x 32, SWIZZLE_128B tensor map; rows past the list are
//     zero-filled by the TMA unit), 2 warps the bulk copies of the pre-packed weight stage (one contiguous b_hi|b_lo|b_b block
//     per stage): a bulk operation costs its issuing thread ~330 ns whatever its size (profiles/r2_a_probes.md), so the two
//     streams alternate between two threads each;
//   * 8 converter warps read the raw stage (conflict-free: one row per lane of a quarter-warp), apply the prologue (SiLU or
//     the per-row c_new u scale), split, and write the canonical K-major UMMA tiles a_hi | a_lo over the raw stage (in place:
//     a named barrier separates the reads from the writes);
//   * 1 thread issues the 2 x 3 tcgen05.mma.kind::f16 (M = 128, N <= 256, K = 16) of a stage and commits them to the stage
//     barrier, which frees the stage;
//   * 8 epilogue warps (two groups of four, one warp per TMEM lane quadrant) read the accumulator with tcgen05.ld, apply 2^-s
//     and the fused epilogue, write a 128 x 32 output tile into shared memory (SWIZZLE_128B, conflict-free one row per lane)
//     and one thread hands it to the TMA unit (cp.async.bulk.tensor store): address generation, coalescing and clipping at the
//     matrix edge cost no instructions (the per-warp transposition tiles of gemm_tc.cu cost ~530 SASS instructions per 16
//     columns, profiles/r2_c_f16s.md).  Rows between the number of active edges and the end of the last tile are written
//     with don't-care values: every edge-sized workspace array holds the full capacity.
//   * rows may be (edge, m) pairs of one irrep inside an [e][comp][c] tensor (tp_big.cuh): tiles then hold d3 * floor(128 / d3)
//     rows and the mapped operand is a 3-D tensor map (c, m, e).
// Two accumulators of 256 columns alternate between consecutive tiles of a CTA.
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstring>

#include "gemm.cuh"
#include "tc_common.cuh"

namespace allegro {
namespace {

constexpr int F_M = 128, F_KS = 32, F_NT = 256, F_S = 3;
constexpr int F_PROD = 4, F_CVT = 8, F_EPI = 8;
constexpr int F_W_MMA = F_PROD, F_W_CVT0 = F_PROD + 1, F_W_EPI0 = F_W_CVT0 + F_CVT;
constexpr int F_T = (F_PROD + 1 + F_CVT + F_EPI) * 32;                 // 672 threads
constexpr uint32_t F_RAW_BYTES = F_M * F_KS * 4;                        // fp32 A stage as loaded
constexpr uint32_t F_CVT_BYTES = F_M * F_KS * 2;                        // one of a_hi / a_lo (they replace the raw stage)
constexpr uint32_t F_BMAX_BYTES = F_NT * F_KS * 2;                      // one of b_hi / b_lo / b_b at 256 columns
constexpr uint32_t F_OFF_B = F_RAW_BYTES;
constexpr uint32_t F_STAGE_BYTES = F_OFF_B + 3 * F_BMAX_BYTES;          // 64 KB
constexpr int F_BAR_CVT = 3;                                            // named barrier of the converter warps (1, 2: epilogue groups)
constexpr uint32_t F_OUT_BYTES = F_M * 32 * 4;                          // one 128 x 32 fp32 output tile per epilogue group
constexpr size_t F_SMEM = (size_t)F_S * F_STAGE_BYTES + 2 * F_OUT_BYTES + 1024;

struct FArgs {
  GemmArgs a;
  const uint8_t* Bp;        // packed b_hi | b_lo | b_b weight stages per column tile
  const float* out_scale;   // 2^-s of this weight matrix (device scalar written by k_pack_scale)
  unsigned long long* trace;   // developer build only
  const float* WgT;         // EPI_GATHER2: transposed species columns [2S][N]
  int Npad, Kpad, n_nt;     // N padded to 16, K to 32, number of column tiles
  int nk0, nk;              // K stages that read A0, total
  int passes;               // 3 = full split, 2 = activations split only, 1 = plain fp16 (precision study)
  int rpt;                  // rows per tile: 128, or d3 * (128 / d3) when rows are (edge, m) pairs of a mapped operand
  int a_d3, c_d3;           // > 0: A0 / C is the 3-D mapped tensor
};

// Developer build (-DF16S_TRACE, ALLEGRO_F16S_TRACE=1 at build time): CTA 0 sums the cycles each role spends in its waits and the
// host prints them per tile after every launch (profiles/r2_c_f16s.md).
#ifdef F16S_TRACE
#define TR_DECL uint64_t tr_w[4] = {0, 0, 0, 0}; const uint64_t tr_t0 = clock64();
#define TR_WAIT(i, stmt) { const uint64_t t_ = clock64(); stmt; tr_w[i] += clock64() - t_; }
#define TR_FLUSH(base) if (blockIdx.x == 0) { for (int i_ = 0; i_ < 4; ++i_) fa.trace[(base) + i_] = tr_w[i_]; fa.trace[(base) + 4] = clock64() - tr_t0; }
#else
#define TR_DECL
#define TR_WAIT(i, stmt) { stmt; }
#define TR_FLUSH(base) {}
#endif

// bounded wait: a protocol error ends in a trap (sticky CUDA error) instead of a hung GPU
__device__ __forceinline__ void mbar_wait_l(uint64_t* bar, uint32_t parity, int line) {
  uint32_t done = 0;
  for (uint32_t it = 0; !done; ++it) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity), "r"(1000u)
        : "memory");
    if (it > (1u << 22)) {
#ifdef F16S_DBGWAIT
      printf("[f16s] wait timed out: line %d block %d warp %d parity %u\n", line, (int)blockIdx.x, (int)(threadIdx.x >> 5), parity);
#endif
      __trap();
    }
  }
}
#define mbar_wait_b(bar, parity) mbar_wait_l(bar, parity, __LINE__)
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(dst)),
               "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(dst)),
               "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tm, int c0, int c1, const void* src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* tm, int c0, int c1, int c2, const void* src) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(src))
               : "memory");
}
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate));
}
// x -> (a_hi, a_lo): a_hi = fp16(x), a_lo = bf16(x - a_hi)
__device__ __forceinline__ void split8(const float (&v)[8], uint4& hi, uint4& lo) {
  uint32_t h[4], l[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const __half2 hh = __floats2half2_rn(v[2 * j], v[2 * j + 1]);
    const float2 hf = __half22float2(hh);
    const __nv_bfloat162 ll = __floats2bfloat162_rn(v[2 * j] - hf.x, v[2 * j + 1] - hf.y);
    h[j] = *reinterpret_cast<const uint32_t*>(&hh);
    l[j] = *reinterpret_cast<const uint32_t*>(&ll);
  }
  hi = make_uint4(h[0], h[1], h[2], h[3]);
  lo = make_uint4(l[0], l[1], l[2], l[3]);
}

// max |w| of the matrix as raw bits (non-negative floats order like their bit patterns)
__global__ void k_pack_absmax(const float* __restrict__ W, int ldw, int wtrans, int N, int K, uint32_t* __restrict__ mx) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  uint32_t v = 0;
  if (idx < (int64_t)N * K) {
    const int n = (int)(idx / K), k = (int)(idx - (int64_t)n * K);
    v = __float_as_uint(fabsf(wtrans ? W[(int64_t)k * ldw + n] : W[(int64_t)n * ldw + k]));
  }
  for (int o = 16; o; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0 && v) atomicMax(mx, v);
}
// sc[0] = 2^s with max |w| 2^s in [2^13, 2^14), sc[1] = 2^-s
__global__ void k_pack_scale(const uint32_t* __restrict__ mx, float* __restrict__ sc) {
  const float m = __uint_as_float(*mx);
  int e = 0, s = 0;
  if (m > 0.f && m < 3.0e38f) { frexpf(m, &e); s = min(max(14 - e, -60), 60); }
  sc[0] = ldexpf(1.f, s);
  sc[1] = ldexpf(1.f, -s);
}
// packed B: per column tile t (n0 = 256 t, Nt columns), per K stage c: [b_hi: Nt x 32 fp16 | b_lo: Nt x 32 fp16 | b_b: Nt x 32 bf16],
// each in the canonical K-major no-swizzle UMMA layout [n/8][k/8][n%8][k%8] (core matrix = 8 rows x 16 bytes; LBO 128 B, SBO 512 B)
__global__ void k_pack_w16(const float* __restrict__ W, int ldw, int wtrans, int N, int K, int Npad, int Kpad, const float* __restrict__ sc,
                           uint8_t* __restrict__ out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)Npad * Kpad) return;
  const int n = (int)(idx / Kpad), k = (int)(idx - (int64_t)n * Kpad);
  float v = 0.f;
  if (n < N && k < K) v = (wtrans ? W[(int64_t)k * ldw + n] : W[(int64_t)n * ldw + k]) * sc[0];
  const __half hi = __float2half_rn(v);
  const __half lo = __float2half_rn(v - __half2float(hi));
  const __nv_bfloat16 bb = __float2bfloat16_rn(v);
  const int tile = n / F_NT, nl = n - tile * F_NT, Nt = min(Npad - tile * F_NT, F_NT);
  const int c = k / F_KS, kl = k - c * F_KS;
  const size_t base = (size_t)tile * F_NT * Kpad * 6 + (size_t)c * Nt * (F_KS * 6);
  const int off = (nl >> 3) * 512 + (kl >> 3) * 128 + (nl & 7) * 16 + (kl & 7) * 2;
  const size_t arr = (size_t)Nt * (F_KS * 2);
  *reinterpret_cast<__half*>(out + base + off) = hi;
  *reinterpret_cast<__half*>(out + base + arr + off) = lo;
  *reinterpret_cast<__nv_bfloat16*>(out + base + 2 * arr + off) = bb;
}

__global__ void __launch_bounds__(F_T, 1) k_gemm_f16s(const __grid_constant__ FArgs fa, const __grid_constant__ CUtensorMap tmA0,
                                                       const __grid_constant__ CUtensorMap tmA1, const __grid_constant__ CUtensorMap tmC,
                                                       const __grid_constant__ CUtensorMap tmC2) {
  extern __shared__ uint8_t smem_dyn[];
  __shared__ __align__(8) uint64_t raw_full[F_S], cvt_full[F_S], mma_done[F_S];
  __shared__ __align__(8) uint64_t acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;
  const GemmArgs& a = fa.a;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint8_t* smem = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);   // SWIZZLE_128B tiles need 1024-byte alignment
  uint8_t* out_tiles = smem + (size_t)F_S * F_STAGE_BYTES;
  const int64_t M = *a.Mptr * a.m_mul;
  const int rpt = fa.rpt;
  const int64_t n_mt = (M + rpt - 1) / rpt;
  const int64_t n_tiles = n_mt * fa.n_nt;
  const int nk = fa.nk;
  const int passes = fa.passes;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 32) {
    for (int s = 0; s < F_S; ++s) {
      mbar_init(&raw_full[s], 1); mbar_init(&cvt_full[s], F_CVT + 1);   // the converter warps + the weight copy: one wait per stage for the issuing thread
      mbar_init(&mma_done[s], 1);
    }
    for (int b = 0; b < 2; ++b) { mbar_init(&acc_full[b], 1); mbar_init(&acc_empty[b], F_EPI); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_d0 = tmem_base_s;

  if (warp < 2) {
    // ---- A producer: TMA loads of the raw fp32 stages, the two warps take alternate stages
    if (lane == 0) {
      const uint32_t a0_bytes = fa.a_d3 ? (uint32_t)rpt * (F_KS * 4) : F_RAW_BYTES;
      const int epb = fa.a_d3 ? rpt / fa.a_d3 : 0;                      // edges per tile of the mapped operand
      uint32_t it = 0;
      TR_DECL
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int mt = (int)(tile / fa.n_nt);
        for (int ks = 0; ks < nk; ++ks, ++it) {
          if ((int)(it & 1) != warp) continue;
          const uint32_t slot = it % F_S, ph = (it / F_S) & 1;
          TR_WAIT(0, mbar_wait_b(&mma_done[slot], ph ^ 1))   // the MMAs that read the converted tile of this slot are complete
          uint8_t* dst = smem + (size_t)slot * F_STAGE_BYTES;
          if (ks < fa.nk0) {
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&raw_full[slot])), "r"(a0_bytes) : "memory");
            if (fa.a_d3) tma_load_3d(dst, &tmA0, ks * F_KS, 0, mt * epb, &raw_full[slot]);
            else tma_load_2d(dst, &tmA0, ks * F_KS, mt * rpt, &raw_full[slot]);
          } else {
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&raw_full[slot])), "r"(F_RAW_BYTES) : "memory");
            tma_load_2d(dst, &tmA1, (ks - fa.nk0) * F_KS, mt * rpt, &raw_full[slot]);
          }
        }
      }
      if (warp == 0) TR_FLUSH(8)
    }
  } else if (warp < 4) {
    // ---- B producer: one bulk copy per stage (hi | lo block of this column tile)
    if (lane == 0) {
      const int w = warp - 2;
      uint32_t it = 0;
      TR_DECL
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int nt = (int)(tile % fa.n_nt);
        const int Nt = min(fa.Npad - nt * F_NT, F_NT);
        const uint8_t* tb = fa.Bp + (size_t)nt * F_NT * fa.Kpad * 6;
        for (int ks = 0; ks < nk; ++ks, ++it) {
          if ((int)(it & 1) != w) continue;
          const uint32_t slot = it % F_S, ph = (it / F_S) & 1;
          TR_WAIT(0, mbar_wait_b(&mma_done[slot], ph ^ 1))
          bulk_g2s(smem + (size_t)slot * F_STAGE_BYTES + F_OFF_B, tb + (size_t)ks * Nt * (F_KS * 6), (uint32_t)Nt * (F_KS * 6), &cvt_full[slot]);
        }
      }
      if (w == 0) TR_FLUSH(16)
    }
  } else if (warp == F_W_MMA) {
    // ---- MMA issuer
    if (lane == 0) {
      uint32_t it = 0, titer = 0;
      TR_DECL
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++titer) {
        const int nt = (int)(tile % fa.n_nt);
        const int Nt = min(fa.Npad - nt * F_NT, F_NT);
        // D fp32 (bit 4), A format at bit 7 / B format at bit 10 (0 = fp16, 1 = bf16), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
        const uint32_t idesc = (1u << 4) | ((uint32_t)(Nt >> 3) << 17) | ((uint32_t)(F_M >> 4) << 24);
        const uint32_t idesc_bb = idesc | (1u << 7) | (1u << 10);
        const uint32_t ab = titer & 1, tmem_d = tmem_d0 + ab * F_NT;
        TR_WAIT(0, mbar_wait_b(&acc_empty[ab], ((titer >> 1) & 1) ^ 1))
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        for (int ks = 0; ks < nk; ++ks, ++it) {
          const uint32_t slot = it % F_S, ph = (it / F_S) & 1;
          TR_WAIT(1, mbar_wait_b(&cvt_full[slot], ph))
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint32_t sbase = smem_u32(smem + (size_t)slot * F_STAGE_BYTES);
          const uint32_t sa_hi = sbase, sa_lo = sa_hi + F_CVT_BYTES;
          const uint32_t sb_hi = sbase + F_OFF_B, sb_lo = sb_hi + (uint32_t)Nt * (F_KS * 2), sb_b = sb_lo + (uint32_t)Nt * (F_KS * 2);
#pragma unroll
          for (int k2 = 0; k2 < F_KS / 16; ++k2) {
            const uint32_t koff = k2 * 256;                     // two 128-byte core-matrix columns per K = 16 step
            const uint64_t dAh = umma_desc(sa_hi + koff, 128, 512), dAl = umma_desc(sa_lo + koff, 128, 512);
            const uint64_t dBh = umma_desc(sb_hi + koff, 128, 512), dBl = umma_desc(sb_lo + koff, 128, 512), dBb = umma_desc(sb_b + koff, 128, 512);
            const uint32_t acc = (ks > 0 || k2 > 0) ? 1u : 0u;
            umma_f16(tmem_d, dAh, dBh, idesc, acc);
            if (passes >= 3) umma_f16(tmem_d, dAh, dBl, idesc, 1u);
            if (passes >= 2) umma_f16(tmem_d, dAl, dBb, idesc_bb, 1u);
          }
          umma_commit(&mma_done[slot]);
        }
        umma_commit(&acc_full[ab]);
      }
      TR_FLUSH(0)
    }
  } else if (warp < F_W_EPI0) {
    // ---- converters: raw fp32 stage -> prologue -> a_hi / a_lo canonical tiles, in place.  Lane l of a warp: rows
    // 16 cw + 8 i + (l & 7) (i = 0, 1), k chunk q = l >> 3 (8 elements): a quarter-warp reads 8 rows of one chunk pair (8 distinct
    // swizzled positions) and writes 128 contiguous bytes.
    const int cw = warp - F_W_CVT0;
    const int q = lane >> 3, r7 = lane & 7;
    uint32_t it = 0;
    TR_DECL
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      const int64_t row0 = (tile / fa.n_nt) * rpt;
      float sc[2] = {1.f, 1.f};
      if (a.pro == PRO_SCALE_U) {
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const int64_t row = row0 + 16 * cw + 8 * i + r7;
          sc[i] = row < M ? a.c_new * a.geo[row * GEO_W + 4] : 0.f;
        }
      }
      for (int ks = 0; ks < nk; ++ks, ++it) {
        const uint32_t slot = it % F_S, ph = (it / F_S) & 1;
        uint8_t* st = smem + (size_t)slot * F_STAGE_BYTES;
        TR_WAIT(0, mbar_wait_b(&raw_full[slot], ph))
        float4 raw[2][2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const uint8_t* rp = st + (16 * cw + 8 * i + r7) * 128;
          raw[i][0] = *reinterpret_cast<const float4*>(rp + (((2 * q) ^ r7) << 4));
          raw[i][1] = *reinterpret_cast<const float4*>(rp + (((2 * q + 1) ^ r7) << 4));
        }
        TR_WAIT(1, asm volatile("bar.sync %0, %1;" ::"n"(F_BAR_CVT), "n"(F_CVT * 32) : "memory"))   // every converter has read its part of the raw stage
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const int r = 16 * cw + 8 * i + r7;
          float v[8] = {raw[i][0].x, raw[i][0].y, raw[i][0].z, raw[i][0].w, raw[i][1].x, raw[i][1].y, raw[i][1].z, raw[i][1].w};
          if (a.pro == PRO_SILU) {
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = silu_f(v[e]);
          } else if (a.pro == PRO_SCALE_U) {
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] *= sc[i];
          }
          uint4 hi, lo;
          split8(v, hi, lo);
          const uint32_t off = (uint32_t)(r >> 3) * 512 + q * 128 + r7 * 16;
          *reinterpret_cast<uint4*>(st + off) = hi;
          *reinterpret_cast<uint4*>(st + F_CVT_BYTES + off) = lo;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy stores -> visible to the tensor core
        __syncwarp();
        if (lane == 0) mbar_arrive(&cvt_full[slot]);
      }
    }
    if (cw == 0 && lane == 0) TR_FLUSH(24)
  } else {
    // ---- epilogue: two groups of four warps (TMEM lane quadrant = warp % 4); a group takes alternate 32-column steps, builds
    // the 128 x 32 output tile in shared memory (row per lane, 16-byte chunks XOR-swizzled like the tensor map) and TMA-stores it.
    const int ew = warp - F_W_EPI0;
    const int quad = warp & 3, grp = ew >> 2;
    const int erow = quad * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(quad * 32) << 16;
    uint8_t* obuf = out_tiles + (size_t)grp * F_OUT_BYTES;
    uint8_t* orow = obuf + erow * 128;
    const int sw = erow & 7;
    const bool leader = (quad == 0 && lane == 0);            // issues the stores of its group
    const int bar_id = 1 + grp;
    const int epb_c = fa.c_d3 ? rpt / fa.c_d3 : 0;
    const int npass = (a.epi == EPI_Y_X || a.epi == EPI_RESIDUAL) ? 2 : 1;
    const float osc = *fa.out_scale;
    uint32_t titer = 0;
    TR_DECL
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++titer) {
      const int mt = (int)(tile / fa.n_nt), nt = (int)(tile % fa.n_nt);
      const int col0 = nt * F_NT, Nt = min(fa.Npad - col0, F_NT);
      const int64_t row0 = (int64_t)mt * rpt, row = row0 + erow;
      const bool row_ok = row < M && erow < rpt;
      float u = 0.f; int zi = 0, zj = 0;
      if (row_ok && a.geo && a.m_mul == 1) {
        const float* gq = a.geo + row * GEO_W;
        u = gq[4]; zi = __float_as_int(gq[6]); zj = __float_as_int(gq[7]);
      }
      const float* xrow = ((a.epi == EPI_ACCUM) ? a.C + row * a.ldc : a.aux + row * a.ldaux);
      const float cu = a.c_new * u;
      const uint32_t ab = titer & 1, tmem_d = tmem_d0 + ab * F_NT;
      TR_WAIT(0, mbar_wait_b(&acc_full[ab], (titer >> 1) & 1))
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
      for (int c32 = grp; c32 * 32 < Nt; c32 += 2) {
        const int nb = col0 + c32 * 32;                          // first global column of this step
        const bool to_c2 = a.epi == EPI_SPLIT_RES && nb >= a.split;
        const int xlim = a.epi == EPI_SPLIT_RES ? a.split : a.N;
        const bool need_x = a.epi == EPI_DSILU || a.epi == EPI_ACCUM || (a.epi == EPI_SPLIT_RES && !to_c2);
#pragma unroll 1
        for (int pass = 0; pass < npass; ++pass) {
          // the previous store of this group has finished reading the tile
          TR_WAIT(1, if (leader) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"))
          TR_WAIT(2, asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory"))
#pragma unroll
          for (int sub = 0; sub < 2; ++sub) {
            const int n0 = c32 * 32 + sub * 16, ng = col0 + n0;
            float v[16];
            tmem_ld16(tmem_d + lane_addr + (uint32_t)n0, v);
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] *= osc;
            float4 x[4];
            const bool ldx = (need_x || (a.epi == EPI_RESIDUAL && pass == 1)) && row_ok;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              x[j] = make_float4(0.f, 0.f, 0.f, 0.f);
              if (ldx && ng + 4 * j < xlim) x[j] = *reinterpret_cast<const float4*>(xrow + ng + 4 * j);
            }
            float4 o[4];
#define F_V(j) make_float4(v[4 * (j)], v[4 * (j) + 1], v[4 * (j) + 2], v[4 * (j) + 3])
            switch (a.epi) {
              case EPI_GATHER2: {
                const float* g1p = fa.WgT + (int64_t)zi * a.N;
                const float* g2p = fa.WgT + (int64_t)(a.S + zj) * a.N;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  const int nn = min(ng + 4 * j, a.N - 4);        // padded columns read a valid address; the store clips them
                  const float4 g1 = *reinterpret_cast<const float4*>(g1p + nn);
                  const float4 g2 = *reinterpret_cast<const float4*>(g2p + nn);
                  const float4 t = F_V(j);
                  o[j] = make_float4(t.x + (g1.x + g2.x), t.y + (g1.y + g2.y), t.z + (g1.z + g2.z), t.w + (g1.w + g2.w));
                }
              } break;
              case EPI_Y_X:
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  const float4 t = F_V(j);
                  o[j] = pass == 0 ? t : make_float4(u * t.x, u * t.y, u * t.z, u * t.w);
                }
                break;
              case EPI_RESIDUAL:
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  const float4 t = F_V(j);
                  o[j] = pass == 0 ? t
                                   : make_float4(a.c_old * x[j].x + cu * t.x, a.c_old * x[j].y + cu * t.y, a.c_old * x[j].z + cu * t.z,
                                                 a.c_old * x[j].w + cu * t.w);
                }
                break;
              case EPI_DSILU:
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  const float4 t = F_V(j);
                  o[j] = make_float4(t.x * dsilu_f(x[j].x), t.y * dsilu_f(x[j].y), t.z * dsilu_f(x[j].z), t.w * dsilu_f(x[j].w));
                }
                break;
              case EPI_ACCUM:
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  const float4 t = F_V(j);
                  o[j] = make_float4(x[j].x + t.x, x[j].y + t.y, x[j].z + t.z, x[j].w + t.w);
                }
                break;
              case EPI_SPLIT_RES:
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                  const float4 t = F_V(j);
                  o[j] = to_c2 ? t : make_float4(a.c_old * x[j].x + t.x, a.c_old * x[j].y + t.y, a.c_old * x[j].z + t.z, a.c_old * x[j].w + t.w);
                }
                break;
              default:
#pragma unroll
                for (int j = 0; j < 4; ++j) o[j] = F_V(j);
                break;
            }
#undef F_V
#pragma unroll
            for (int j = 0; j < 4; ++j) *reinterpret_cast<float4*>(orow + (((sub * 4 + j) ^ sw) << 4)) = o[j];
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // tile stores -> visible to the TMA unit
          TR_WAIT(3, asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory"))
          if (leader) {
            const bool second = to_c2 || pass == 1;
            const CUtensorMap* tm = second ? &tmC2 : &tmC;
            const int cc = to_c2 ? nb - a.split : nb;
            if (fa.c_d3 && !second) tma_store_3d(tm, cc, 0, mt * epb_c, obuf);
            else tma_store_2d(tm, cc, (int)row0, obuf);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
          }
        }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(&acc_empty[ab]);
    }
    if (leader) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // all stores complete before the CTA retires
    if (leader && grp == 0) TR_FLUSH(32)
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d0), "r"(512));
  }
}

// ---- host side -------------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
    cudaGetLastError();
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// fp32 matrix [rows][K] with leading dimension ld, boxes of 32 columns x 128 rows, SWIZZLE_128B, zero fill / clipping outside.
// d3 > 0: rows are (edge, m) pairs of one irrep of an [e][comp][c] tensor (A points at its first row): 3-D map (c, m, e) with
// boxes of 32 x d3 x (128 / d3); od = comps per edge.  box_rows < 128 for the plain side of a mapped GEMM: a store must not
// touch the rows of the next tile.
bool make_map(Model* m, const float* A, int K, int ld, int64_t rows, int d3, int od, int box_rows, CUtensorMap* out) {
  const std::array<int64_t, 6> key = {(int64_t)(uintptr_t)A, K, ld, rows, d3 + 16 * box_rows, od};
  auto it = m->tmaps.find(key);
  if (it != m->tmaps.end()) { std::memcpy(out, &it->second, sizeof(CUtensorMap)); return true; }
  EncodeTiledFn enc = encode_fn();
  if (!enc) return false;
  CUtensorMap tm;
  CUresult r;
  if (d3 > 0) {
    cuuint64_t gdim[3] = {(cuuint64_t)K, (cuuint64_t)d3, (cuuint64_t)(rows / d3)};
    cuuint64_t gstr[2] = {(cuuint64_t)ld * 4, (cuuint64_t)od * ld * 4};
    cuuint32_t box[3] = {(cuuint32_t)F_KS, (cuuint32_t)d3, (cuuint32_t)(F_M / d3)};
    cuuint32_t estr[3] = {1, 1, 1};
    r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(A), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  } else {
    cuuint64_t gdim[2] = {(cuuint64_t)K, (cuuint64_t)rows};
    cuuint64_t gstr[1] = {(cuuint64_t)ld * 4};
    cuuint32_t box[2] = {(cuuint32_t)F_KS, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(A), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  if (r != CUDA_SUCCESS) return false;
  TMapStore s;
  static_assert(sizeof(TMapStore) == sizeof(CUtensorMap), "tensor map storage");
  std::memcpy(&s, &tm, sizeof(tm));
  if (m->tmaps.size() > 4096) m->tmaps.clear();   // workspace reallocations leave dead entries behind
  m->tmaps[key] = s;
  std::memcpy(out, &tm, sizeof(tm));
  return true;
}

// packed weights of a call site; the last 256 bytes of the buffer hold {2^s, 2^-s, max |w| bits}
uint8_t* packed_weights16(Model* m, const GemmArgs& a, cudaStream_t st, int* Npad_out, int* Kpad_out, const float** out_scale) {
  const int K = a.K0 + a.K1;
  const int Npad = (a.N + 15) / 16 * 16, Kpad = (K + F_KS - 1) / F_KS * F_KS;
  *Npad_out = Npad; *Kpad_out = Kpad;
  const size_t bytes = 6 * (size_t)Npad * Kpad;
  const std::array<int64_t, 5> key = {(int64_t)(a.W - m->d_w), a.ldw, a.wtrans | 16, a.N, K};
  auto it = m->packed_w.find(key);
  if (it != m->packed_w.end()) {
    *out_scale = reinterpret_cast<const float*>(reinterpret_cast<uint8_t*>(it->second) + bytes) + 1;
    return reinterpret_cast<uint8_t*>(it->second);
  }
  float* Bp = nullptr;
  if (cudaMalloc(&Bp, bytes + 256) != cudaSuccess) { cudaGetLastError(); m->err = "packed weight allocation failed"; return nullptr; }
  uint8_t* B8 = reinterpret_cast<uint8_t*>(Bp);
  float* sc = reinterpret_cast<float*>(B8 + bytes);
  cudaMemsetAsync(sc, 0, 256, st);
  const int64_t nw = (int64_t)a.N * K, tot = (int64_t)Npad * Kpad;
  k_pack_absmax<<<(unsigned)((nw + 255) / 256), 256, 0, st>>>(a.W, a.ldw, a.wtrans, a.N, K, reinterpret_cast<uint32_t*>(sc + 2));
  k_pack_scale<<<1, 1, 0, st>>>(reinterpret_cast<const uint32_t*>(sc + 2), sc);
  k_pack_w16<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(a.W, a.ldw, a.wtrans, a.N, K, Npad, Kpad, sc, B8);
  m->packed_w[key] = Bp;
  *out_scale = sc + 1;
  return B8;
}

}  // namespace

// packed b_hi | b_lo | b_b stages of a weight matrix (cached per call site) and its 2^-s, for tp_mix.cu
const uint8_t* f16s_packed_weights(Model* m, const GemmArgs& a, cudaStream_t st, const float** out_scale) {
  int Npad = 0, Kpad = 0;
  return packed_weights16(m, a, st, &Npad, &Kpad, out_scale);
}

// Returns false when the shape / alignment is outside what the kernel takes (the caller then uses k_gemm_tc).
bool launch_gemm_f16s(Model* m, const GemmArgs& a, int64_t m_cap, cudaStream_t st) {
  const int K = a.K0 + a.K1;
  auto al = [](const void* p) { return ((uintptr_t)p & 15) == 0; };
  if (K < 1 || a.N < 4 || a.N % 4 || a.lda0 % 4 || !al(a.A0)) return false;
  if (a.K1 > 0 && (a.K0 % F_KS || a.lda1 % 4 || !al(a.A1))) return false;
  if (a.ldc % 4 || !al(a.C)) return false;
  if (a.C2 && (a.ldc2 % 4 || !al(a.C2))) return false;
  if (a.aux && (a.ldaux % 4 || !al(a.aux))) return false;
  if (a.epi == EPI_SPLIT_RES && a.split % 32) return false;
  if (a.m_mul != 1 && (a.epi != EPI_STORE || a.pro != PRO_NONE)) return false;
  if ((a.amap_d3 || a.cmap_d3) && (a.K1 > 0 || a.epi != EPI_STORE)) return false;
  if (a.amap_d3 && a.cmap_d3 && a.amap_d3 != a.cmap_d3) return false;
  if (m->f16_rows_cap <= 0) return false;
  FArgs fa{};
  fa.a = a;
  fa.passes = m->f16_passes;
  uint8_t* Bp = packed_weights16(m, a, st, &fa.Npad, &fa.Kpad, &fa.out_scale);
  if (!Bp) return false;
  fa.Bp = Bp;
  fa.n_nt = (fa.Npad + F_NT - 1) / F_NT;
  fa.nk0 = (a.K0 + F_KS - 1) / F_KS;
  fa.nk = fa.nk0 + (a.K1 + F_KS - 1) / F_KS;
  fa.WgT = nullptr;
  if (a.epi == EPI_GATHER2) {
    fa.WgT = transposed_species_columns(m, a, st);
    if (!fa.WgT) return false;
  }
  const int d3 = a.amap_d3 ? a.amap_d3 : a.cmap_d3;
  fa.rpt = d3 ? d3 * (F_M / d3) : F_M;
  fa.a_d3 = a.amap_d3; fa.c_d3 = a.cmap_d3;
  const int64_t rows_cap = m->f16_rows_cap * a.m_mul;                              // rows the operand buffers hold (workspace capacity)
  CUtensorMap t0, t1, tc, tc2;
  if (a.amap_d3) { if (!make_map(m, a.A0 + (int64_t)a.amap_off * a.lda0, a.K0, a.lda0, rows_cap, a.amap_d3, a.amap_od, F_M, &t0)) return false; }
  else if (!make_map(m, a.A0, a.K0, a.lda0, rows_cap, 0, 0, F_M, &t0)) return false;
  if (a.K1 > 0) { if (!make_map(m, a.A1, a.K1, a.lda1, rows_cap, 0, 0, F_M, &t1)) return false; }
  else t1 = t0;
  const int cw = a.epi == EPI_SPLIT_RES ? a.split : a.N;
  if (a.cmap_d3) { if (!make_map(m, a.C + (int64_t)a.cmap_off * a.ldc, cw, a.ldc, rows_cap, a.cmap_d3, a.cmap_od, F_M, &tc)) return false; }
  else if (!make_map(m, a.C, cw, a.ldc, rows_cap, 0, 0, fa.rpt, &tc)) return false;
  if (a.C2) { if (!make_map(m, a.C2, a.epi == EPI_SPLIT_RES ? a.N - a.split : a.N, a.ldc2, rows_cap, 0, 0, fa.rpt, &tc2)) return false; }
  else tc2 = tc;
  static int attr_dev = -1;
  if (attr_dev != m->device) {
    if (cudaFuncSetAttribute(k_gemm_f16s, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM) != cudaSuccess) { cudaGetLastError(); return false; }
    attr_dev = m->device;
  }
  const int64_t tiles = ((m_cap * a.m_mul + fa.rpt - 1) / fa.rpt) * fa.n_nt;
  const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(tiles, m->num_sms));
#ifdef F16S_TRACE
  static unsigned long long* d_trace = nullptr;
  if (!d_trace) cudaMalloc(&d_trace, 64 * sizeof(unsigned long long));
  cudaMemsetAsync(d_trace, 0, 64 * sizeof(unsigned long long), st);
  fa.trace = d_trace;
#endif
  prof_begin(m, st, KC_GEMM16, 2.0 * a.N * K * a.m_mul);
  k_gemm_f16s<<<grid, F_T, F_SMEM, st>>>(fa, t0, t1, tc, tc2);
  prof_end(m, st);
#ifdef F16S_TRACE
  {
    unsigned long long h[64];
    cudaStreamSynchronize(st);
    cudaMemcpy(h, d_trace, sizeof(h), cudaMemcpyDeviceToHost);
    const double nt = (double)std::max<int64_t>(1, (tiles + grid - 1) / grid);
    std::printf("[f16s trace] K=%d N=%d pro=%d epi=%d tiles/CTA=%.0f stages=%d | per tile: mma total %.0f (acc_empty %.0f cvt_full %.0f b_full %.0f) | "
                "A-prod wait %.0f | B-prod wait %.0f | cvt total %.0f (raw_full %.0f bar %.0f) | epi total %.0f (acc_full %.0f store-read %.0f bar1 %.0f bar2 %.0f)\n",
                K, a.N, a.pro, a.epi, nt, fa.nk, h[4] / nt, h[0] / nt, h[1] / nt, h[2] / nt, h[8] / nt, h[16] / nt, h[28] / nt, h[24] / nt, h[25] / nt,
                h[36] / nt, h[32] / nt, h[33] / nt, h[34] / nt, h[35] / nt);
  }
#endif
  m->launches += 1;
  return true;
}

}  // namespace allegro
