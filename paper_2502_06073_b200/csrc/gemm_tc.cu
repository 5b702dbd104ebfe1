// gemm_tc.cu — the edge-by-width GEMMs of the network on the 5th-generation tensor cores (tcgen05, sm_100a).
//
// Same contract as k_gemm (gemm.cuh): C[e, n] = epi( sum_k pro(A[e, k]) B(k, n) ) with the fused prologues and
// epilogues, for the dense linears of PAPER.md:93 / Table 1 (two-body MLP, W_init / W_env, latent MLPs and their
// transposes in the backward pass).
//
// Precision: north_star allows tensor cores "only in a precision that stays inside the stated tolerance"
// (forces within 1e-4 x RMS against fp64).  A single kind::tf32 pass (2^-11 per operand) does not; the 3-pass split
//   a = a_hi + a_lo (a_hi = rna-rounded TF32),  A B ~= A_hi B_hi + A_hi B_lo + A_lo B_hi   (fp32 accumulation in TMEM)
// leaves ~2^-21 relative error per product, the same class as fp32 FMA.
//
// Structure of one CTA (128 threads, one 128-row tile of edges x up to 128 output columns):
//   * the four warps stage a 128 x 32 slice of A (prologue applied, split into hi/lo) and the matching N x 32 slice of B
//     (weights, split into hi/lo) in shared memory in the canonical K-major no-swizzle UMMA layout
//     [row/8][k/4][row%8][k%4] (core matrix = 8 rows x 16 B; LBO = 128 B between the k-chunks, SBO = 1024 B between
//     8-row groups), two stages;
//   * one elected thread issues 3 x 4 tcgen05.mma.cta_group::1.kind::tf32 (M=128, N, K=8) per slice and commits them to
//     the stage's mbarrier, so the next slice is staged while the tensor pipe runs;
//   * accumulators live in TMEM (N fp32 columns x 128 lanes); the epilogue reads them with tcgen05.ld.32x32b (one
//     output row per thread) and applies the fused epilogue while writing to global memory.
#include <cstdint>

#include "gemm.cuh"

namespace allegro {
namespace {

constexpr int TC_M = 128, TC_KC = 32, TC_T = 128, TC_NMAX = 128;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ float tf32_rna(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

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
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
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

// smem layout per stage: A_hi | A_lo (128 x 32 fp32 each = 16 KB) | B_hi | B_lo (Npad x 32 fp32 each)
__global__ void __launch_bounds__(TC_T) k_gemm_tc(GemmArgs a, int Npad, int tmem_cols) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t mbar[2];
  __shared__ uint32_t tmem_base_s;
  const int64_t M = *a.Mptr;
  const int64_t row0 = (int64_t)blockIdx.x * TC_M;
  if (row0 >= M) return;
  const int col0 = blockIdx.y * TC_NMAX;
  const int Nt = min(Npad - col0, TC_NMAX);           // columns of this tile (multiple of 16)
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K = a.K0 + a.K1;
  const int nchunks = (K + TC_KC - 1) / TC_KC;
  const uint32_t a_bytes = TC_M * TC_KC * 4, b_bytes = (uint32_t)Nt * TC_KC * 4;
  const uint32_t stage_bytes = 2 * a_bytes + 2 * b_bytes;
  uint8_t* sm = smem_raw;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(tmem_cols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    mbar_init(&mbar[0], 1); mbar_init(&mbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_d = tmem_base_s;
  // instruction descriptor: D fp32, A/B tf32, K-major both, N, M=128
  const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(Nt >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);

  const int64_t arow = row0 + tid;                    // this thread stages row `tid` of A and column `tid` of B
  const bool arow_ok = arow < M;
  float ascale = 1.f;
  if (a.pro == PRO_SCALE_U && arow_ok) ascale = a.c_new * a.geo[arow * GEO_W + 4];
  const int bn = col0 + tid;
  const bool bcol_ok = tid < Nt && bn < a.N;

  for (int c = 0; c < nchunks; ++c) {
    const int b = c & 1;
    if (c >= 2) mbar_wait(&mbar[b], (uint32_t)(((c >> 1) - 1) & 1));   // MMAs of slice c-2 have drained stage b
    uint8_t* st = sm + (size_t)b * stage_bytes;
    float* Ahi = reinterpret_cast<float*>(st);
    float* Alo = reinterpret_cast<float*>(st + a_bytes);
    float* Bhi = reinterpret_cast<float*>(st + 2 * a_bytes);
    float* Blo = reinterpret_cast<float*>(st + 2 * a_bytes + b_bytes);
    const int k0 = c * TC_KC;
    // ---- A slice: row `tid`, 8 quads of k
    {
      const int off_row = (tid >> 3) * (TC_KC / 4) * 32 + (tid & 7) * 4;   // floats: (row/8)*SBO + (row%8)*16B
#pragma unroll
      for (int q = 0; q < TC_KC / 4; ++q) {
        const int kk = k0 + q * 4;
        float v[4] = {0.f, 0.f, 0.f, 0.f};
        if (arow_ok && kk < K) {
          const float* src; int kl, kmax;
          if (kk < a.K0) { src = a.A0 + arow * a.lda0; kl = kk; kmax = a.K0; }
          else { src = a.A1 + arow * a.lda1; kl = kk - a.K0; kmax = a.K1; }
          if (kl + 3 < kmax && ((((uintptr_t)(src + kl)) & 15) == 0)) {
            const float4 t = *reinterpret_cast<const float4*>(src + kl);
            v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
          } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int kq = kk + e;
              if (kq < K) v[e] = (kq < a.K0) ? a.A0[arow * a.lda0 + kq] : a.A1[arow * a.lda1 + (kq - a.K0)];
            }
          }
          if (a.pro == PRO_SILU) {
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] = silu_f(v[e]);
          } else if (a.pro == PRO_SCALE_U) {
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] *= ascale;
          }
        }
        float4 hi, lo;
        hi.x = tf32_rna(v[0]); hi.y = tf32_rna(v[1]); hi.z = tf32_rna(v[2]); hi.w = tf32_rna(v[3]);
        lo.x = v[0] - hi.x; lo.y = v[1] - hi.y; lo.z = v[2] - hi.z; lo.w = v[3] - hi.w;
        *reinterpret_cast<float4*>(Ahi + off_row + q * 32) = hi;
        *reinterpret_cast<float4*>(Alo + off_row + q * 32) = lo;
      }
    }
    // ---- B slice: output column `tid` (B is K-major: rows = n, contiguous along k)
    if (tid < Nt) {
      const int off_row = (tid >> 3) * (TC_KC / 4) * 32 + (tid & 7) * 4;
#pragma unroll
      for (int q = 0; q < TC_KC / 4; ++q) {
        float v[4] = {0.f, 0.f, 0.f, 0.f};
        if (bcol_ok) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int kk = k0 + q * 4 + e;
            if (kk < K) v[e] = a.wtrans ? a.W[(int64_t)kk * a.ldw + bn] : a.W[(int64_t)bn * a.ldw + kk];
          }
        }
        float4 hi, lo;
        hi.x = tf32_rna(v[0]); hi.y = tf32_rna(v[1]); hi.z = tf32_rna(v[2]); hi.w = tf32_rna(v[3]);
        lo.x = v[0] - hi.x; lo.y = v[1] - hi.y; lo.z = v[2] - hi.z; lo.w = v[3] - hi.w;
        *reinterpret_cast<float4*>(Bhi + off_row + q * 32) = hi;
        *reinterpret_cast<float4*>(Blo + off_row + q * 32) = lo;
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy smem writes -> visible to the tensor core
    __syncthreads();
    if (tid == 0) {
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t sa_hi = smem_u32(Ahi), sa_lo = smem_u32(Alo), sb_hi = smem_u32(Bhi), sb_lo = smem_u32(Blo);
      const int ksteps = min(TC_KC, (K - k0 + 7) / 8 * 8) / 8;   // K=8 steps that hold real data
      const uint32_t sbo = (TC_KC / 4) * 128;   // bytes between 8-row groups
      for (int ks = 0; ks < ksteps; ++ks) {
        const uint32_t koff = ks * 256;          // two 128-byte k-chunks per K=8 step
        const uint64_t dAh = umma_desc(sa_hi + koff, 128, sbo), dAl = umma_desc(sa_lo + koff, 128, sbo);
        const uint64_t dBh = umma_desc(sb_hi + koff, 128, sbo), dBl = umma_desc(sb_lo + koff, 128, sbo);
        umma_tf32(tmem_d, dAl, dBh, idesc, (c > 0 || ks > 0) ? 1u : 0u);   // small terms first
        umma_tf32(tmem_d, dAh, dBl, idesc, 1u);
        umma_tf32(tmem_d, dAh, dBh, idesc, 1u);
      }
      umma_commit(&mbar[b]);
    }
  }
  // all slices issued: wait for the last commit (commits complete in order)
  {
    const int c = nchunks - 1;
    mbar_wait(&mbar[c & 1], (uint32_t)((c >> 1) & 1));
  }
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

  // ---- epilogue: thread -> output row (TMEM lane 32*warp + lane)
  const int64_t row = row0 + tid;
  float u = 0.f; int zi = 0, zj = 0;
  if (row < M) {
    if (a.epi == EPI_Y_X || a.epi == EPI_RESIDUAL) u = a.geo[row * GEO_W + 4];
    if (a.epi == EPI_GATHER2) { zi = __float_as_int(a.geo[row * GEO_W + 6]); zj = __float_as_int(a.geo[row * GEO_W + 7]); }
  }
  for (int n0 = 0; n0 < Nt; n0 += 16) {
    float v[16];
    tmem_ld16(tmem_d + ((uint32_t)(warp * 32) << 16) + (uint32_t)n0, v);
    if (row < M) {
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int n = col0 + n0 + j;
        if (n < a.N) gemm_epi(a, row, n, v[j], u, zi, zj);
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"(tmem_cols));
  }
}

}  // namespace

void launch_gemm_tc(Model* m, const GemmArgs& a, int64_t m_cap, cudaStream_t st) {
  const int Npad = (a.N + 15) / 16 * 16;
  const int Nt = std::min(Npad, TC_NMAX);
  int tmem_cols = 32;
  while (tmem_cols < Nt) tmem_cols *= 2;
  const size_t smem = 2 * (size_t)(2 * TC_M * TC_KC * 4 + 2 * Nt * TC_KC * 4);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(k_gemm_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (2 * TC_M * TC_KC * 4 + 2 * TC_NMAX * TC_KC * 4));
    attr_set = true;
  }
  dim3 grid((unsigned)((m_cap + TC_M - 1) / TC_M), (unsigned)((Npad + TC_NMAX - 1) / TC_NMAX));
  prof_begin(m, st, KC_GEMM, 2.0 * a.N * (a.K0 + a.K1));
  k_gemm_tc<<<grid, TC_T, smem, st>>>(a, Npad, tmem_cols);
  prof_end(m, st);
  m->launches += 1;
}

}  // namespace allegro
