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
// Structure of one CTA (256 threads, one 128-row tile of edges x up to 128 output columns; three CTAs fit on an SM):
//   * B (the weight block) is split into hi/lo and laid out in the canonical K-major no-swizzle UMMA layout ONCE per
//     call site (k_pack_w, cached in the handle); per 16-deep k slice one thread pulls its 2 x N x 16 block into shared
//     memory with a single cp.async.bulk that completes on the stage's mbarrier;
//   * the eight warps stage the 128 x 16 slice of A (prologue applied, hi/lo split) in the same canonical layout
//     [row/8][k/4][row%8][k%4] (core matrix = 8 rows x 16 B; LBO = 128 B between k-chunks, SBO = 512 B between 8-row
//     groups), two stages;
//   * one elected thread issues 3 x 2 tcgen05.mma.cta_group::1.kind::tf32 (M=128, N, K=8) per slice and commits them to
//     the stage's mbarrier, so the next slice is staged while the tensor pipe runs;
//   * accumulators live in TMEM (N fp32 columns x 128 lanes); the epilogue reads them with tcgen05.ld.32x32b (one
//     output row per thread, two warps per lane quadrant taking alternate 16-column groups) and applies the fused
//     epilogue with 128-bit stores.
#include <cstdint>
#include <cstdio>
#include <cstdlib>

#include "gemm.cuh"
#include "tc_common.cuh"

namespace allegro {
namespace {

constexpr int TC_M = 128, TC_KC = 16, TC_T = 256, TC_NMAX = 256;   // one CTA: 128 rows x up to 256 columns (256 TMEM columns)

// Packed B operand: for each 128-column tile, for each k slice: [hi block | lo block], block = Nt x 16 fp32 canonical.
__global__ void k_pack_w(const float* __restrict__ W, int ldw, int wtrans, int N, int K, int Npad, int Kpad, float* __restrict__ out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)Npad * Kpad) return;
  const int n = (int)(idx / Kpad), k = (int)(idx - (int64_t)n * Kpad);
  float v = 0.f;
  if (n < N && k < K) v = wtrans ? W[(int64_t)k * ldw + n] : W[(int64_t)n * ldw + k];
  const float hi = tf32_rna(v), lo = v - hi;
  const int tile = n / TC_NMAX, nl = n - tile * TC_NMAX, Nt = min(Npad - tile * TC_NMAX, TC_NMAX);
  const int c = k / TC_KC, kl = k - c * TC_KC;
  const int64_t base = (int64_t)tile * TC_NMAX * Kpad * 2 + (int64_t)c * (2 * Nt * TC_KC);
  const int off = (nl >> 3) * (TC_KC / 4) * 32 + (kl >> 2) * 32 + (nl & 7) * 4 + (kl & 3);
  out[base + off] = hi;
  out[base + Nt * TC_KC + off] = lo;
}

// smem per stage: A_hi | A_lo (128 x 16 fp32 each = 8 KB) | B_hi | B_lo (Nt x 16 fp32 each)
__global__ void __launch_bounds__(TC_T + 32) k_gemm_tc(GemmArgs a, const float* __restrict__ Bp, int Npad, int Kpad, int tmem_cols, int vec_ok,
                                                       int passes) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t mbar_mma[2];
  __shared__ __align__(8) uint64_t mbar_b[2];
  __shared__ __align__(8) uint64_t mbar_staged[2];         // A staging buffer written by the 8 compute warps
  __shared__ uint32_t tmem_base_s;
  const int64_t M = *a.Mptr * a.m_mul;
  const int64_t row0 = (int64_t)blockIdx.x * TC_M;
  if (row0 >= M) return;
  const int col0 = blockIdx.y * TC_NMAX;
  const int Nt = min(Npad - col0, TC_NMAX);           // columns of this tile (multiple of 16)
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K = a.K0 + a.K1;
  const int nchunks = Kpad / TC_KC;
  constexpr uint32_t a_bytes = TC_M * TC_KC * 4;
  const uint32_t b_bytes = (uint32_t)Nt * TC_KC * 4;
  const uint32_t stage_bytes = 2 * a_bytes + 2 * b_bytes;
  const float* Bt = Bp + (int64_t)blockIdx.y * TC_NMAX * Kpad * 2;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(tmem_cols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    mbar_init(&mbar_mma[0], 1); mbar_init(&mbar_mma[1], 1);
    mbar_init(&mbar_b[0], 1); mbar_init(&mbar_b[1], 1);
    mbar_init(&mbar_staged[0], 8); mbar_init(&mbar_staged[1], 8);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_d = tmem_base_s;
  // instruction descriptor: D fp32 (bit 4), A/B tf32 (2 at bits 7 and 10), both K-major, N>>3 at bit 17, M>>4 at bit 24
  const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(Nt >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);

  if (warp == 8) {
    // weight loader + MMA issuer (one thread): the compute warps never wait behind the tensor-core queue
    if (lane == 0) {
      for (int c = 0; c < nchunks; ++c) {
        const int b = c & 1;
        if (c >= 2) mbar_wait(&mbar_mma[b], (uint32_t)(((c >> 1) - 1) & 1));   // slice c-2 done: stage b (A and B) is free
        uint8_t* st = smem_raw + (size_t)b * stage_bytes;
        float* Bhi = reinterpret_cast<float*>(st + 2 * a_bytes);
        bulk_g2s(Bhi, Bt + (int64_t)c * (2 * Nt * TC_KC), 2 * b_bytes, &mbar_b[b]);
        mbar_wait(&mbar_staged[b], (uint32_t)((c >> 1) & 1));
        mbar_wait(&mbar_b[b], (uint32_t)((c >> 1) & 1));
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t sa_hi = smem_u32(st), sa_lo = sa_hi + a_bytes, sb_hi = smem_u32(Bhi), sb_lo = sb_hi + b_bytes;
        constexpr uint32_t sbo = (TC_KC / 4) * 128;                   // bytes between 8-row groups
#pragma unroll
        for (int ks = 0; ks < TC_KC / 8; ++ks) {
          const uint32_t koff = ks * 256;                              // two 128-byte k-chunks per K=8 step
          const uint64_t dAh = umma_desc(sa_hi + koff, 128, sbo), dAl = umma_desc(sa_lo + koff, 128, sbo);
          const uint64_t dBh = umma_desc(sb_hi + koff, 128, sbo), dBl = umma_desc(sb_lo + koff, 128, sbo);
          const uint32_t acc = (c > 0 || ks > 0) ? 1u : 0u;
          if (passes >= 2) umma_tf32(tmem_d, dAl, dBh, idesc, acc);   // small terms first
          if (passes >= 3) umma_tf32(tmem_d, dAh, dBl, idesc, 1u);
          umma_tf32(tmem_d, dAh, dBh, idesc, passes >= 2 ? 1u : acc);
        }
        umma_commit(&mbar_mma[b]);
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    return;
  }
  const int r = tid & 127, qh = tid >> 7;              // this thread stages row r, k-quads 2*qh and 2*qh+1 of each slice
  const bool arow_ok = row0 + r < M;
  const int64_t arow = a.amap_d3 ? ((row0 + r) / a.amap_d3) * a.amap_od + a.amap_off + (row0 + r) % a.amap_d3 : row0 + r;
  float ascale = 1.f;
  if (a.pro == PRO_SCALE_U && arow_ok) ascale = a.c_new * a.geo[arow * GEO_W + 4];
  const int off_row = (r >> 3) * (TC_KC / 4) * 32 + (r & 7) * 4;   // floats: (row/8)*SBO + (row%8)*16 B

  // raw A values of one 16-deep slice (this thread: row r, k-quads 2*qh and 2*qh+1), no prologue applied yet
  auto load_slice = [&](int c, float (&v)[2][4]) {
#pragma unroll
    for (int qq = 0; qq < 2; ++qq) {
      const int kk = c * TC_KC + (qh * 2 + qq) * 4;
#pragma unroll
      for (int e = 0; e < 4; ++e) v[qq][e] = 0.f;
      if (arow_ok && kk < K) {
        const float* src; int kl, kmax;
        if (kk < a.K0) { src = a.A0 + arow * a.lda0; kl = kk; kmax = a.K0; }
        else { src = a.A1 + arow * a.lda1; kl = kk - a.K0; kmax = a.K1; }
        if (kl + 3 < kmax && ((((uintptr_t)(src + kl)) & 15) == 0)) {
          const float4 t = *reinterpret_cast<const float4*>(src + kl);
          v[qq][0] = t.x; v[qq][1] = t.y; v[qq][2] = t.z; v[qq][3] = t.w;
        } else {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int kq = kk + e;
            if (kq < K) v[qq][e] = (kq < a.K0) ? a.A0[arow * a.lda0 + kq] : a.A1[arow * a.lda1 + (kq - a.K0)];
          }
        }
      }
    }
  };
  float vcur[2][4], vnext[2][4];
  load_slice(0, vcur);
  for (int c = 0; c < nchunks; ++c) {
    const int b = c & 1;
    if (c + 1 < nchunks) load_slice(c + 1, vnext);                        // in flight while slice c is staged and issued
    if (c >= 2) mbar_wait(&mbar_mma[b], (uint32_t)(((c >> 1) - 1) & 1));   // MMAs of slice c-2 have drained stage b
    uint8_t* st = smem_raw + (size_t)b * stage_bytes;
    float* Ahi = reinterpret_cast<float*>(st);
    float* Alo = reinterpret_cast<float*>(st + a_bytes);
#pragma unroll
    for (int qq = 0; qq < 2; ++qq) {
      const int q = qh * 2 + qq;
      float v[4] = {vcur[qq][0], vcur[qq][1], vcur[qq][2], vcur[qq][3]};
      if (a.pro == PRO_SILU) {
#pragma unroll
        for (int e = 0; e < 4; ++e) v[e] = silu_f(v[e]);
      } else if (a.pro == PRO_SCALE_U) {
#pragma unroll
        for (int e = 0; e < 4; ++e) v[e] *= ascale;
      }
      float4 hi, lo;
      hi.x = tf32_trunc(v[0]); hi.y = tf32_trunc(v[1]); hi.z = tf32_trunc(v[2]); hi.w = tf32_trunc(v[3]);   // see k_gemm_chain
      lo.x = v[0] - hi.x; lo.y = v[1] - hi.y; lo.z = v[2] - hi.z; lo.w = v[3] - hi.w;
      *reinterpret_cast<float4*>(Ahi + off_row + q * 32) = hi;
      *reinterpret_cast<float4*>(Alo + off_row + q * 32) = lo;
    }
#pragma unroll
    for (int qq = 0; qq < 2; ++qq)
#pragma unroll
      for (int e = 0; e < 4; ++e) vcur[qq][e] = vnext[qq][e];
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy smem writes -> visible to the tensor core
    __syncwarp();
    if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&mbar_staged[b])) : "memory");
  }
  {   // all slices issued: wait for the last commit (commits complete in order)
    const int c = nchunks - 1;
    mbar_wait(&mbar_mma[c & 1], (uint32_t)((c >> 1) & 1));
  }
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

  // ---- epilogue: thread -> output row (TMEM lane quadrant = warp % 4), warps w and w+4 alternate 16-column groups
  const int quad = warp & 3, half = warp >> 2;
  const int64_t row = row0 + quad * 32 + lane;
  float u = 0.f; int zi = 0, zj = 0;
  if (row < M) {
    if (a.epi == EPI_Y_X || a.epi == EPI_RESIDUAL) u = a.geo[row * GEO_W + 4];
    if (a.epi == EPI_GATHER2) { zi = __float_as_int(a.geo[row * GEO_W + 6]); zj = __float_as_int(a.geo[row * GEO_W + 7]); }
  }
  for (int n0 = half * 16; n0 < Nt; n0 += 32) {
    float v[16];
    tmem_ld16(tmem_d + ((uint32_t)(quad * 32) << 16) + (uint32_t)n0, v);
    if (row < M) {
      if (vec_ok) {
        const int nb = col0 + n0;
        const bool aux_kind = a.epi == EPI_DSILU || a.epi == EPI_RESIDUAL || a.epi == EPI_ACCUM || (a.epi == EPI_SPLIT_RES && nb + 16 <= a.split);
        if (aux_kind) {
          // the four auxiliary loads of a 16-column step are issued together (one basic block), then the arithmetic, then the
          // stores: the per-group form waits for one global load at a time (42 % of the warp-state samples of this kernel,
          // profiles/r1_h_gemm_tc.md).  Columns past N read a clamped valid address and are not stored.
          const float* xs = (a.epi == EPI_ACCUM) ? a.C + row * a.ldc : a.aux + row * a.ldaux;
          float4 x[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) x[j] = *reinterpret_cast<const float4*>(xs + min(nb + 4 * j, a.N - 4));
          float4 o1[4], o2[4];
          const float cu = a.c_new * u;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 t = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
            o1[j] = t; o2[j] = t;
            if (a.epi == EPI_DSILU) o1[j] = make_float4(t.x * dsilu_f(x[j].x), t.y * dsilu_f(x[j].y), t.z * dsilu_f(x[j].z), t.w * dsilu_f(x[j].w));
            else if (a.epi == EPI_ACCUM) o1[j] = make_float4(x[j].x + t.x, x[j].y + t.y, x[j].z + t.z, x[j].w + t.w);
            else if (a.epi == EPI_RESIDUAL)
              o2[j] = make_float4(a.c_old * x[j].x + cu * t.x, a.c_old * x[j].y + cu * t.y, a.c_old * x[j].z + cu * t.z, a.c_old * x[j].w + cu * t.w);
            else o1[j] = make_float4(a.c_old * x[j].x + t.x, a.c_old * x[j].y + t.y, a.c_old * x[j].z + t.z, a.c_old * x[j].w + t.w);
          }
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int n = nb + 4 * j;
            if (n < a.N) {
              *reinterpret_cast<float4*>(a.C + row * a.ldc + n) = o1[j];
              if (a.epi == EPI_RESIDUAL) *reinterpret_cast<float4*>(a.C2 + row * a.ldc2 + n) = o2[j];
            }
          }
        } else {
#pragma unroll
          for (int j = 0; j < 16; j += 4) {
            const int n = col0 + n0 + j;
            if (n < a.N) gemm_epi4(a, row, n, make_float4(v[j], v[j + 1], v[j + 2], v[j + 3]), u, zi, zj);
          }
        }
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int n = col0 + n0 + j;
          if (n < a.N) gemm_epi(a, row, n, v[j], u, zi, zj);
        }
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

float* packed_weights(Model* m, const GemmArgs& a, cudaStream_t st, int* Npad_out, int* Kpad_out) {
  const int K = a.K0 + a.K1;
  const int Npad = (a.N + 15) / 16 * 16, Kpad = (K + TC_KC - 1) / TC_KC * TC_KC;
  *Npad_out = Npad; *Kpad_out = Kpad;
  const std::array<int64_t, 5> key = {(int64_t)(a.W - m->d_w), a.ldw, a.wtrans, a.N, K};
  auto it = m->packed_w.find(key);
  if (it != m->packed_w.end()) return it->second;
  float* Bp = nullptr;
  if (cudaMalloc(&Bp, sizeof(float) * 2 * (size_t)Npad * Kpad) != cudaSuccess) { cudaGetLastError(); m->err = "packed weight allocation failed"; return nullptr; }
  const int64_t tot = (int64_t)Npad * Kpad;
  k_pack_w<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(a.W, a.ldw, a.wtrans, a.N, K, Npad, Kpad, Bp);
  m->packed_w[key] = Bp;
  return Bp;
}

void launch_gemm_tc(Model* m, const GemmArgs& a, int64_t m_cap, cudaStream_t st) {
  const int K = a.K0 + a.K1;
  int Npad, Kpad;
  float* Bp = packed_weights(m, a, st, &Npad, &Kpad);
  if (!Bp) return;
  const int Nt = std::min(Npad, TC_NMAX);
  int tmem_cols = 32;
  while (tmem_cols < Nt) tmem_cols *= 2;
  const size_t smem = 2 * (size_t)(2 * TC_M * TC_KC * 4 + 2 * Nt * TC_KC * 4);
  static int attr_dev = -1;   // the attribute is per device
  if (attr_dev != m->device) {
    cudaFuncSetAttribute(k_gemm_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (2 * TC_M * TC_KC * 4 + 2 * TC_NMAX * TC_KC * 4));
    attr_dev = m->device;
  }
  auto al = [](const void* p) { return ((uintptr_t)p & 15) == 0; };
  int vec_ok = (a.N % 4 == 0) && (a.ldc % 4 == 0) && al(a.C);
  if (a.C2) vec_ok = vec_ok && (a.ldc2 % 4 == 0) && al(a.C2);
  if (a.aux) vec_ok = vec_ok && (a.ldaux % 4 == 0) && al(a.aux);
  if (a.epi == EPI_SPLIT_RES) vec_ok = vec_ok && (a.split % 4 == 0);
  dim3 grid((unsigned)((m_cap + TC_M - 1) / TC_M), (unsigned)((Npad + TC_NMAX - 1) / TC_NMAX));
  prof_begin(m, st, KC_GEMM, 2.0 * a.N * K * a.m_mul);
  k_gemm_tc<<<grid, TC_T + 32, smem, st>>>(a, Bp, Npad, Kpad, tmem_cols, vec_ok, m->f16_passes);
  prof_end(m, st);
  m->launches += 1;
}

}  // namespace allegro

// =============================================================================================================
// Chained GEMMs: up to CH_MAX dependent linears of one MLP on the same 128-row tile of edges.  The activation never
// leaves the SM between stages: the epilogue of stage s reads the accumulator from TMEM, applies its fused epilogue
// (global stores of what the backward pass needs), applies the prologue of stage s+1 and writes the fp32 result to the
// activation columns of TMEM; in the k loop the compute warps read it back 16 columns at a time, split it hi/lo and stage
// it in the canonical K-major UMMA layout, a loader warp streams the pre-packed weight slices with cp.async.bulk
// (CH_NB slots) and an issuer warp issues the MMAs.  Details above k_gemm_chain and in DESIGN.md section 6.
// =============================================================================================================
namespace allegro {
namespace {

constexpr int CH_MAX = 4, CH_NB = 3, CH_KMAX = 128, CH_NMAX = 128, CH_T = TC_T + 64;   // 8 compute warps + weight-loader warp + MMA-issuer warp

struct ChainArgs {
  int n;
  int passes;                    // 3 = hi*hi + hi*lo + lo*hi (default); 2 / 1 only for the precision study (R4)
  GemmArgs st[CH_MAX];
  const float* Bp[CH_MAX];
  const float* WgT[CH_MAX];      // EPI_GATHER2: species columns of W transposed, [2S][N]
  int Npad[CH_MAX], Kpad[CH_MAX];
};

__global__ void k_transpose_wg(const float* __restrict__ Wg, int ldwg, int S, int N, float* __restrict__ out) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * (int64_t)S * N) return;
  const int z = (int)(idx / N), n = (int)(idx - (int64_t)z * N);
  out[idx] = Wg[(int64_t)n * ldwg + z];
}

__device__ __forceinline__ bool epi_needs_aux(const GemmArgs& a, int n) {
  return a.epi == EPI_RESIDUAL || a.epi == EPI_DSILU || a.epi == EPI_ACCUM || (a.epi == EPI_SPLIT_RES && n < a.split);
}
// TMEM: columns [0, 128) accumulator D, columns [128, 256) the activation that feeds the current stage (fp32, prologue
// already applied).  Shared memory: two 16-deep A staging buffers (hi | lo, canonical layout; reused as the per-warp
// transposition tiles of the epilogue) and CH_NB weight slots filled by a dedicated loader warp.
__global__ void __launch_bounds__(CH_T, 2) k_gemm_chain(const __grid_constant__ ChainArgs ca) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t mbar_s[CH_NB];          // slice g done (barrier g % CH_NB, phase g / CH_NB): frees A buffer and weight slot
  __shared__ __align__(8) uint64_t mbar_b[CH_NB];          // weight slot landed
  __shared__ __align__(8) uint64_t mbar_staged[2];         // A staging buffer b written by all 8 compute warps
  __shared__ uint32_t tmem_base_s;
  __shared__ float dot_s[TC_M];
  const int64_t M = *ca.st[0].Mptr;
  const int64_t row0 = (int64_t)blockIdx.x * TC_M;
  if (row0 >= M) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  constexpr uint32_t a_floats = TC_M * TC_KC, slot_floats = 2 * CH_NMAX * TC_KC;
  float* As = reinterpret_cast<float*>(smem_raw);          // [2][hi | lo]
  float* Bs = As + 2 * 2 * a_floats;                        // [CH_NB][hi | lo]

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(256));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    for (int i = 0; i < CH_NB; ++i) { mbar_init(&mbar_b[i], 1); mbar_init(&mbar_s[i], 1); }
    mbar_init(&mbar_staged[0], 8); mbar_init(&mbar_staged[1], 8);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  if (warp == 8) {
    // weight loader: streams the pre-packed slices of every stage through the CH_NB slots, never blocking the issuer
    if (lane == 0) {
      int g = 0;
      for (int s = 0; s < ca.n; ++s) {
        const int Ntl = ca.Npad[s], nch = ca.Kpad[s] / TC_KC;
        for (int c = 0; c < nch; ++c, ++g) {
          const int slot = g % CH_NB, use = g / CH_NB;
          if (use > 0) mbar_wait(&mbar_s[slot], (uint32_t)((use - 1) & 1));   // slice g - CH_NB used this slot
          bulk_g2s(Bs + slot * slot_floats, ca.Bp[s] + (int64_t)c * (2 * Ntl * TC_KC), (uint32_t)(2 * Ntl * TC_KC * 4), &mbar_b[slot]);
        }
      }
    }
    __syncthreads();   // matches the block-wide barrier before the TMEM release
    return;
  }
  if (warp == 9) {
    // MMA issuer: the only thread that talks to the tensor core.  It waits for a staged A slice (8 warp arrivals) and its
    // weight slot, issues the 3 x 2 MMAs and commits them to the slice barrier; the compute warps never wait on it.
    if (lane == 0) {
      const uint32_t tmem_dd = tmem_base_s;
      int g = 0;
      for (int s = 0; s < ca.n; ++s) {
        const int Nt = ca.Npad[s], nch = ca.Kpad[s] / TC_KC;
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(Nt >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);
        const uint32_t b_bytes = (uint32_t)Nt * TC_KC * 4;
        for (int c = 0; c < nch; ++c, ++g) {
          const int b = g & 1, slot = g % CH_NB, use = g / CH_NB;
          mbar_wait(&mbar_staged[b], (uint32_t)((g >> 1) & 1));
          mbar_wait(&mbar_b[slot], (uint32_t)(use & 1));
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint32_t sa_hi = smem_u32(As + b * 2 * a_floats), sa_lo = sa_hi + a_floats * 4;
          const uint32_t sb_hi = smem_u32(Bs + slot * slot_floats), sb_lo = sb_hi + b_bytes;
          constexpr uint32_t sbo = (TC_KC / 4) * 128;
#pragma unroll
          for (int ks = 0; ks < TC_KC / 8; ++ks) {
            const uint32_t koff = ks * 256;
            const uint64_t dAh = umma_desc(sa_hi + koff, 128, sbo), dAl = umma_desc(sa_lo + koff, 128, sbo);
            const uint64_t dBh = umma_desc(sb_hi + koff, 128, sbo), dBl = umma_desc(sb_lo + koff, 128, sbo);
            const uint32_t acc = (c > 0 || ks > 0) ? 1u : 0u;
            if (ca.passes >= 2) umma_tf32(tmem_dd, dAl, dBh, idesc, acc);
            if (ca.passes >= 3) umma_tf32(tmem_dd, dAh, dBl, idesc, 1u);
            umma_tf32(tmem_dd, dAh, dBh, idesc, ca.passes >= 2 ? 1u : acc);
          }
          umma_commit(&mbar_s[slot]);
        }
      }
    }
    __syncthreads();
    return;
  }
  const uint32_t tmem_d = tmem_base_s, tmem_act = tmem_base_s + 128;
  const int quad = warp & 3, half = warp >> 2;
  const int erow = quad * 32 + lane;                       // this thread's row of the tile (TMEM lane)
  const uint32_t lane_addr = (uint32_t)(quad * 32) << 16;
  const int64_t row = row0 + erow, rbase = row0 + quad * 32;
  const bool row_ok = row < M;
  // per-warp tiles: wtile (stores, stage-in) and dtile (prefetched dot operand) inside the A staging area, which is idle during
  // the epilogues; xtile (prefetched auxiliary rows) behind the weight slots, so that it can be filled during the k loop
  float* wtile = As + warp * (2 * 32 * WT_LD);
  float* dtile = wtile + 32 * WT_LD;
  float* xtile = Bs + CH_NB * slot_floats + warp * (32 * WT_LD);
  float u = 0.f; int zi = 0, zj = 0;
  if (row_ok) {
    const float* gq = ca.st[0].geo + row * GEO_W;
    u = gq[4]; zi = __float_as_int(gq[6]); zj = __float_as_int(gq[7]);
  }
  // ---- stage-in: A of the first stage from global memory -> activation columns of TMEM (prologue applied)
  {
    const GemmArgs& a = ca.st[0];
    const int ngrp = ca.Kpad[0] >> 4;
    float ascale = 1.f;
    if (a.pro == PRO_SCALE_U) ascale = a.c_new * u;
    auto ldg_grp = [&](float4 (&t)[4], int k0) {
      if (k0 < a.K0) warp_tile_ldg(t, lane, a.A0, a.lda0, rbase, M, k0, a.K0);
      else warp_tile_ldg(t, lane, a.A1, a.lda1, rbase, M, k0 - a.K0, a.K1);
    };
    auto put_grp = [&](const float4 (&t)[4], int k0) {
      float4 x[4];
      warp_tile_xpose(wtile, t, x, lane);
      if (a.pro == PRO_SILU) {
#pragma unroll
        for (int j = 0; j < 4; ++j) x[j] = make_float4(silu_f(x[j].x), silu_f(x[j].y), silu_f(x[j].z), silu_f(x[j].w));
      } else {
        const float sc = (a.pro == PRO_SCALE_U) ? ascale : 1.f;
#pragma unroll
        for (int j = 0; j < 4; ++j) x[j] = make_float4(x[j].x * sc, x[j].y * sc, x[j].z * sc, x[j].w * sc);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) tmem_st4(tmem_act + lane_addr + (uint32_t)(k0 + 4 * j), x[j]);
    };
    // two 16-column groups per iteration: both global loads are in flight before the first one is consumed
#pragma unroll 1
    for (int gk = half; gk < ngrp; gk += 4) {
      float4 t0[4], t1[4];
      const bool second = gk + 2 < ngrp;
      ldg_grp(t0, gk * 16);
      if (second) ldg_grp(t1, (gk + 2) * 16);
      put_grp(t0, gk * 16);
      if (second) put_grp(t1, (gk + 2) * 16);
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  asm volatile("bar.sync 1, 256;" ::: "memory");
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

  const int off_row = (erow >> 3) * (TC_KC / 4) * 32 + (erow & 7) * 4;
  int gc = 0;                                               // global slice counter
  for (int s = 0; s < ca.n; ++s) {
    const GemmArgs& a = ca.st[s];
    const int Nt = ca.Npad[s], nchunks = ca.Kpad[s] / TC_KC;
    const bool ld_d = a.dot_out && !a.dotv;
    const float* xsrc = (a.epi == EPI_ACCUM) ? a.C : a.aux;
    const int ldx = (a.epi == EPI_ACCUM) ? a.ldc : a.ldaux;
    // auxiliary rows of the first epilogue step: in flight during the whole k loop
    if (epi_needs_aux(a, half * 16)) warp_tile_prefetch(xtile, lane, xsrc, ldx, rbase, M, half * 16, a.N);
    asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll 1
    for (int c = 0; c < nchunks; ++c) {
      const int g = gc + c, b = g & 1;
      if (g >= 2) mbar_wait(&mbar_s[(g - 2) % CH_NB], (uint32_t)(((g - 2) / CH_NB) & 1));   // MMAs of slice g-2 have drained buffer b
      float* Ahi = As + b * 2 * a_floats;
      float* Alo = Ahi + a_floats;
      float v[8];
      tmem_ld8(tmem_act + lane_addr + (uint32_t)(c * TC_KC + half * 8), v);
#pragma unroll
      for (int qq = 0; qq < 2; ++qq) {
        float4 hi, lo;
        // hi = the 19 bits the tensor core reads (truncation: one instruction instead of the four of the emulated cvt.rna);
        // lo = v - hi is exact in fp32 and |lo| < 2^-10 |v|, so hi*hi + hi*lo + lo*hi still carries ~2^-20 per product
        hi.x = tf32_trunc(v[4 * qq]); hi.y = tf32_trunc(v[4 * qq + 1]); hi.z = tf32_trunc(v[4 * qq + 2]); hi.w = tf32_trunc(v[4 * qq + 3]);
        lo.x = v[4 * qq] - hi.x; lo.y = v[4 * qq + 1] - hi.y; lo.z = v[4 * qq + 2] - hi.z; lo.w = v[4 * qq + 3] - hi.w;
        *reinterpret_cast<float4*>(Ahi + off_row + (half * 2 + qq) * 32) = hi;
        *reinterpret_cast<float4*>(Alo + off_row + (half * 2 + qq) * 32) = lo;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // this thread's stores -> visible to the tensor core
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&mbar_staged[b])) : "memory");
    }
    gc += nchunks;
    {   // every slice issued: both staging buffers must have drained before they serve as transposition tiles
      const int g = gc - 1;
      mbar_wait(&mbar_s[g % CH_NB], (uint32_t)((g / CH_NB) & 1));
      if (g >= 1) mbar_wait(&mbar_s[(g - 1) % CH_NB], (uint32_t)(((g - 1) / CH_NB) & 1));
    }
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    // ---- epilogue of stage s; the value the next stage consumes goes back to TMEM with that stage's prologue applied
    const bool last = (s + 1 == ca.n);
    const int npro = last ? PRO_NONE : ca.st[s + 1].pro;
    const float nscale = (!last && npro == PRO_SCALE_U) ? ca.st[s + 1].c_new * u : 1.f;
    const bool two = (a.epi == EPI_Y_X || a.epi == EPI_RESIDUAL);
    float dacc = 0.f;
    if (ld_d) warp_tile_prefetch(dtile, lane, a.dotB, a.lddot, rbase, M, half * 16, a.N);
    asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll 1
    for (int n0 = half * 16; n0 < Nt; n0 += 32) {
      float4 x[4], o1[4], yd[4];
      {   // this step's auxiliary row segments were prefetched; the next step's are requested before the arithmetic
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 4; ++j) { x[j] = make_float4(0.f, 0.f, 0.f, 0.f); yd[j] = x[j]; }
        if (ld_d) warp_tile_read(dtile, yd, lane);
        if (epi_needs_aux(a, n0)) warp_tile_read(xtile, x, lane);
        __syncwarp();
        const int n1 = n0 + 32;
        if (n1 < Nt) {
          if (ld_d) warp_tile_prefetch(dtile, lane, a.dotB, a.lddot, rbase, M, n1, a.N);
          if (epi_needs_aux(a, n1)) warp_tile_prefetch(xtile, lane, xsrc, ldx, rbase, M, n1, a.N);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
      }
      float v[16];
      tmem_ld16(tmem_d + lane_addr + (uint32_t)n0, v);
      // The epilogue kind is resolved once per 16-column step (not per 4-column group), so that each phase below is one
      // basic block over all 16 values and the scheduler can overlap their dependency chains.
      float4 p[4];                                           // what the next stage / the row dot product consumes
#define CH_V(j) make_float4(v[4 * (j)], v[4 * (j) + 1], v[4 * (j) + 2], v[4 * (j) + 3])
      switch (a.epi) {
        case EPI_GATHER2: {
          const float* g1p = ca.WgT[s] + (int64_t)zi * a.N;
          const float* g2p = ca.WgT[s] + (int64_t)(a.S + zj) * a.N;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int nn = min(n0 + 4 * j, a.N - 4);          // padded columns read a valid address; they are masked below
            const float4 g1 = *reinterpret_cast<const float4*>(g1p + nn);
            const float4 g2 = *reinterpret_cast<const float4*>(g2p + nn);
            const float4 t = CH_V(j);
            o1[j] = make_float4(t.x + (g1.x + g2.x), t.y + (g1.y + g2.y), t.z + (g1.z + g2.z), t.w + (g1.w + g2.w));
            p[j] = o1[j];
          }
        } break;
        case EPI_Y_X:
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 t = CH_V(j);
            o1[j] = t; p[j] = make_float4(u * t.x, u * t.y, u * t.z, u * t.w);
          }
          break;
        case EPI_RESIDUAL: {
          const float cu = a.c_new * u;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 t = CH_V(j);
            o1[j] = t;
            p[j] = make_float4(a.c_old * x[j].x + cu * t.x, a.c_old * x[j].y + cu * t.y, a.c_old * x[j].z + cu * t.z, a.c_old * x[j].w + cu * t.w);
          }
        } break;
        case EPI_DSILU:
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 t = CH_V(j);
            o1[j] = make_float4(t.x * dsilu_f(x[j].x), t.y * dsilu_f(x[j].y), t.z * dsilu_f(x[j].z), t.w * dsilu_f(x[j].w));
            p[j] = o1[j];
          }
          break;
        case EPI_ACCUM:
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 t = CH_V(j);
            o1[j] = make_float4(x[j].x + t.x, x[j].y + t.y, x[j].z + t.z, x[j].w + t.w);
            p[j] = o1[j];
          }
          break;
        case EPI_SPLIT_RES: {
          const bool res = n0 < a.split;                      // split % 16 == 0: a step lies on one side
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float4 t = CH_V(j);
            o1[j] = res ? make_float4(a.c_old * x[j].x + t.x, a.c_old * x[j].y + t.y, a.c_old * x[j].z + t.z, a.c_old * x[j].w + t.w) : t;
            p[j] = t;
          }
        } break;
        default:
#pragma unroll
          for (int j = 0; j < 4; ++j) { o1[j] = CH_V(j); p[j] = o1[j]; }
          break;
      }
#undef CH_V
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (!row_ok || n0 + 4 * j >= a.N) p[j] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (a.dot_out) {
        if (a.dotv) {
#pragma unroll
          for (int j = 0; j < 4; ++j) yd[j] = *reinterpret_cast<const float4*>(a.dotv + min(n0 + 4 * j, a.N - 4));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
          dacc = fmaf(p[j].x, yd[j].x, fmaf(p[j].y, yd[j].y, fmaf(p[j].z, yd[j].z, fmaf(p[j].w, yd[j].w, dacc))));
      }
      if (!last) {   // next stage's prologue applied on the way back to TMEM; p itself is still needed for the C2 store
        if (npro == PRO_SILU) {
#pragma unroll
          for (int j = 0; j < 4; ++j)
            tmem_st4(tmem_act + lane_addr + (uint32_t)(n0 + 4 * j), make_float4(silu_f(p[j].x), silu_f(p[j].y), silu_f(p[j].z), silu_f(p[j].w)));
        } else {
          const float sc = (npro == PRO_SCALE_U) ? nscale : 1.f;
#pragma unroll
          for (int j = 0; j < 4; ++j)
            tmem_st4(tmem_act + lane_addr + (uint32_t)(n0 + 4 * j), make_float4(p[j].x * sc, p[j].y * sc, p[j].z * sc, p[j].w * sc));
        }
      }
      // p is zero outside the valid rows / columns, exactly where the tile store is masked: it serves as the C2 operand
      if (a.epi == EPI_SPLIT_RES && n0 >= a.split) {
        warp_tile_store(wtile, o1, lane, a.C2, a.ldc2, rbase, M, n0 - a.split, a.N - a.split);
      } else {
        // the adjoint of a hidden layer is consumed by the next chained stage only: it never goes to global memory
        if (!(a.epi == EPI_DSILU && !last)) warp_tile_store(wtile, o1, lane, a.C, a.ldc, rbase, M, n0, a.epi == EPI_SPLIT_RES ? a.split : a.N);
        if (two) warp_tile_store(wtile, p, lane, a.C2, a.ldc2, rbase, M, n0, a.N);
      }
    }
    if (a.dot_out) {   // the two warps that share a row quadrant combine their halves of the row dot product
      if (half == 1) dot_s[erow] = dacc;
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (half == 0 && row_ok) a.dot_out[row] = (a.dot_accum ? a.dot_out[row] : 0.f) + a.dot_scale * (dacc + dot_s[erow]);
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    asm volatile("bar.sync 1, 256;" ::: "memory");
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"(256));
  }
}

}  // namespace
}  // namespace allegro

namespace allegro {

const float* transposed_species_columns(Model* m, const GemmArgs& a, cudaStream_t st) {
  const std::array<int64_t, 5> key = {(int64_t)(a.Wg - m->d_w), a.ldwg, -7, a.N, a.S};
  auto it = m->packed_w.find(key);
  if (it == m->packed_w.end()) {
    float* T = nullptr;
    if (cudaMalloc(&T, sizeof(float) * 2 * (size_t)a.S * a.N) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    const int64_t tot = 2 * (int64_t)a.S * a.N;
    k_transpose_wg<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(a.Wg, a.ldwg, a.S, a.N, T);
    it = m->packed_w.emplace(key, T).first;
  }
  return it->second;
}

bool launch_gemm_chain(Model* m, const GemmArgs* stages, int n_stages, int64_t m_cap, cudaStream_t st) {
  if (!m->use_tc || !m->use_chain || n_stages < 1 || n_stages > CH_MAX || m_cap <= 0) return false;
  ChainArgs ca{};
  ca.n = n_stages;
  ca.passes = m->f16_passes;
  auto al = [](const void* p) { return ((uintptr_t)p & 15) == 0; };
  double work = 0;
  int nmax = 16;
  for (int s = 0; s < n_stages; ++s) {
    const GemmArgs& a = stages[s];
    const int K = a.K0 + a.K1;
    if (K > CH_KMAX || a.N > CH_NMAX) return false;
    if (s > 0 && (a.K1 != 0 || a.K0 != stages[s - 1].N)) return false;
    // a chained stage reads the previous stage's output from TMEM: it must BE that output (C, or C2 of a two-output epilogue)
    if (s > 0 && a.A0 != stages[s - 1].C && a.A0 != stages[s - 1].C2) return false;
    bool vec_ok = (a.N % 4 == 0) && (a.ldc % 4 == 0) && al(a.C);
    if (a.C2) vec_ok = vec_ok && (a.ldc2 % 4 == 0) && al(a.C2);
    if (a.aux) vec_ok = vec_ok && (a.ldaux % 4 == 0) && al(a.aux);
    if (a.epi == EPI_SPLIT_RES) vec_ok = vec_ok && (a.split % 16 == 0);
    if (a.dot_out && a.dotB) vec_ok = vec_ok && (a.lddot % 4 == 0) && al(a.dotB);
    if (a.dot_out && a.dotv) vec_ok = vec_ok && al(a.dotv);
    if (s == 0) {
      vec_ok = vec_ok && (a.lda0 % 4 == 0) && al(a.A0) && (a.K0 % 4 == 0);
      if (a.K1 > 0) vec_ok = vec_ok && (a.K0 % 16 == 0) && (a.lda1 % 4 == 0) && al(a.A1) && (a.K1 % 4 == 0);
    }
    if (!vec_ok) return false;
  }
  for (int s = 0; s < n_stages; ++s) {
    ca.st[s] = stages[s];
    ca.WgT[s] = nullptr;
    if (stages[s].epi == EPI_GATHER2) {
      ca.WgT[s] = transposed_species_columns(m, stages[s], st);
      if (!ca.WgT[s]) return false;
    }
    ca.Bp[s] = packed_weights(m, stages[s], st, &ca.Npad[s], &ca.Kpad[s]);
    if (!ca.Bp[s]) return false;
    nmax = std::max(nmax, ca.Npad[s]);
    work += 2.0 * stages[s].N * (stages[s].K0 + stages[s].K1);
  }
  (void)nmax;
  // A staging 32 KB + CH_NB weight slots 48 KB + one prefetch tile per compute warp 16 KB = 96 KB: two CTAs per SM
  const size_t smem = (size_t)(2 * 2 * TC_M * TC_KC + CH_NB * 2 * CH_NMAX * TC_KC + 8 * 32 * WT_LD) * sizeof(float);
  static int attr_dev = -1;   // the attribute is per device
  if (attr_dev != m->device) { cudaFuncSetAttribute(k_gemm_chain, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr_dev = m->device; }
  prof_begin(m, st, KC_GEMM, work);
  k_gemm_chain<<<(unsigned)((m_cap + TC_M - 1) / TC_M), CH_T, smem, st>>>(ca);
  prof_end(m, st);
  m->launches += 1;
  return true;
}

}  // namespace allegro
