// tp_mix.cu — F8 + F9 + F11 of one layer in ONE kernel for the many-channel networks (n = 64; Table 1 "64 tensor
// features"): the Clebsch-Gordan tensor product on the CUDA cores feeds the channel-mixing linear on the tensor cores through
// shared memory, so the per-path products T_p[(e, m)][c] (40 KB per edge and layer on BASELINE.json configs[3]) never exist in
// HBM.  Replaces k_tpo_fwd + one k_gemm_f16s launch per output irrep (tp_big.cuh), which wrote and re-read T: 24 GB per layer and
// 600 k-edge chunk, 12 ms of a 90 ms chunk (profiles/r2_d_launches_cfg3.md).
//
//   V^L[e, o, m, c'] = sum_{p in o} sum_c T_p[e, m, c] W_o[c', p n + c],   T_p[e, m, c] = sum_{k1 k2} C_p[k1 k2 m] V[e, k1, c] Gamma[i(e), k2, c]
//
// One persistent CTA per SM, tiles of 16 edges.  Rows of the MMA are (edge, m) pairs of one output irrep (16 d3 <= 112 of 128), its
// columns the 64 output channels; one accumulator D_o of 64 TMEM columns per output irrep (<= 8 irreps = 512 columns).  The K
// dimension of irrep o is (path, channel); it is walked in steps of 32 channels: a tile is processed as two halves (channels
// 0-31, 32-63), and in each half path by path:
//   * 16 compute warps (512 threads, one (edge, channel) pair each, V and Gamma in registers) evaluate the generated coupling code
//     of the path, split the d3 values as in gemm_f16s.cu (a_hi = fp16(t), a_lo = bf16(t - a_hi)) and write them into an A stage
//     in the canonical K-major layout of that kernel (128 rows x 32 k, hi | lo, 16 KB).  Lane mapping: 8 channels x 4 edges per
//     warp, so that the 2-byte stores of a warp fall into 32 distinct banks;
//   * a producer thread streams the weight stage of (path, half) — 64 x 32 of b_hi | b_lo | b_b, 12 KB, exactly one K stage of the
//     packed weights of gemm_f16s.cu — from L2 with one bulk copy;
//   * one thread issues the 2 x 3 tcgen05.mma.kind::f16 (M 128, N 64, K 16) of the step into D_o and commits them to the
//     barriers that free the A stage and the weight slot.
// After the last step the compute warps read the accumulators (one TMEM lane = one (edge, m) row = 64 contiguous output floats),
// apply 2^-s of the weight matrix and store V^L[e][o_off + m][0..63].  F9 (scalar outputs s) is stored by the compute threads.
// Every barrier wait is bounded (trap, not hang).
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <algorithm>

#include "gemm.cuh"
#include "tc_common.cuh"
#include "tp_big.cuh"

namespace allegro {
namespace {

constexpr int X_EDGES = 16, X_N = 64;
constexpr int X_CW = 16;                                  // compute warps
constexpr int X_T = (X_CW + 3) * 32;                      // + MMA warp + two weight-producer warps = 608 threads
constexpr int X_NA = 4, X_NW = 4;                         // A stages = weight slots: ONE commit per step frees both (a tcgen05.commit costs the
                                                          // issuing thread ~200 cycles, measured: two per step made it the bottleneck)
constexpr uint32_t X_A_BYTES = 128 * 32 * 2 * 2;          // a_hi | a_lo, 16 KB
constexpr uint32_t X_W_BYTES = X_N * 32 * 6;              // b_hi | b_lo | b_b, 12 KB
constexpr size_t X_SMEM = (size_t)X_NA * X_A_BYTES + (size_t)X_NW * X_W_BYTES + 1024;

struct XArgs {
  const uint8_t* Bp[TP3_MAXO];       // packed weights of irrep o (gemm_f16s.cu layout, one column tile of 64)
  const float* oscale[TP3_MAXO];     // 2^-s of that matrix
};

__device__ __forceinline__ void x_umma_f16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate));
}
// The six MMAs of one step in one statement.  fa / fb: low descriptor words of the A stage / weight slot; the operands of the
// step sit at fixed offsets from them (in 16-byte units): a_hi +0, a_lo +512 (8 KB), second K = 16 step +16 (256 B);
// b_hi +0, b_lo +256 (4 KB), b_b +512.
__device__ __forceinline__ void x_step_mma(uint32_t d_tmem, uint32_t idesc, uint32_t idesc_bb, uint32_t acc_first, uint32_t hi32, uint32_t fa, uint32_t fb) {
  asm volatile(
      "{\n\t.reg .pred pf, pt;\n\t.reg .b64 ah0, al0, ah1, al1, bh0, bl0, bb0, bh1, bl1, bb1;\n\t.reg .b32 t;\n\t"
      "setp.ne.b32 pf, %3, 0;\n\t"
      "setp.eq.b32 pt, %3, %3;\n\t"
      "mov.b64 ah0, {%5, %4};\n\t"
      "add.u32 t, %5, 512;\n\t mov.b64 al0, {t, %4};\n\t"
      "add.u32 t, %5, 16;\n\t  mov.b64 ah1, {t, %4};\n\t"
      "add.u32 t, %5, 528;\n\t mov.b64 al1, {t, %4};\n\t"
      "mov.b64 bh0, {%6, %4};\n\t"
      "add.u32 t, %6, 256;\n\t mov.b64 bl0, {t, %4};\n\t"
      "add.u32 t, %6, 512;\n\t mov.b64 bb0, {t, %4};\n\t"
      "add.u32 t, %6, 16;\n\t  mov.b64 bh1, {t, %4};\n\t"
      "add.u32 t, %6, 272;\n\t mov.b64 bl1, {t, %4};\n\t"
      "add.u32 t, %6, 528;\n\t mov.b64 bb1, {t, %4};\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], ah0, bh0, %1, pf;\n\t"
#ifndef X_FEWMMA
      "tcgen05.mma.cta_group::1.kind::f16 [%0], ah0, bl0, %1, pt;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], al0, bb0, %2, pt;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], ah1, bh1, %1, pt;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], ah1, bl1, %1, pt;\n\t"
#endif
      "tcgen05.mma.cta_group::1.kind::f16 [%0], al1, bb1, %2, pt;\n\t}"
      ::"r"(d_tmem), "r"(idesc), "r"(idesc_bb), "r"(acc_first), "r"(hi32), "r"(fa), "r"(fb)
      : "memory");
}
// bounded wait without a suspend-time hint: the steps of this kernel are a few hundred cycles long
__device__ __forceinline__ void x_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  for (uint32_t it = 0; !done; ++it) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (it > (1u << 26)) __trap();
  }
}
// a whole warp waits: one lane polls (32 lanes polling one mbarrier are 32 serialised shared-memory operations per round)
__device__ __forceinline__ void x_wait_warp(uint64_t* bar, uint32_t parity, int lane) {
  if (lane == 0) x_wait(bar, parity);
  __syncwarp();
}
__device__ __forceinline__ void x_arrive(uint64_t* bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory"); }

#ifdef X_TRACE
#define XT_DECL unsigned long long xt[4] = {0, 0, 0, 0}; const unsigned long long xt0 = clock64();
#define XT(i, stmt) { const unsigned long long t_ = clock64(); stmt; xt[i] += clock64() - t_; }
#define XT_PRINT(name) if (blockIdx.x == 0) printf("[tpmix %s] sig %d tiles %lld total %llu w0 %llu w1 %llu w2 %llu w3 %llu\n", name, SIG, (long long)((n_tiles + gridDim.x - 1) / gridDim.x), clock64() - xt0, xt[0], xt[1], xt[2], xt[3]);
#else
#define XT_DECL
#define XT(i, stmt) { stmt; }
#define XT_PRINT(name) {}
#endif

template <int SIG>
__global__ void __launch_bounds__(X_T, 1) k_tpmix_fwd(TpLayerDev ly, TpIo io, XArgs xa) {
  using D = tpgen::SigDims<SIG>;
  extern __shared__ uint8_t x_smem_dyn[];
  __shared__ __align__(8) uint64_t a_full[X_NA], st_done[X_NA], acc_full, acc_empty;
  __shared__ uint32_t tmem_base_s;
  __shared__ int n_steps_s;
  __shared__ uint8_t st_o[D::NPATH], st_pidx[D::NPATH];   // the (irrep, path) steps of one half, in the order the compute warps walk them
  uint8_t* smem = x_smem_dyn + ((1024u - (smem_u32(x_smem_dyn) & 1023u)) & 1023u);
  uint8_t* w_ring = smem + (size_t)X_NA * X_A_BYTES;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t M = *io.Mptr;
  const int64_t n_tiles = (M + X_EDGES - 1) / X_EDGES;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 32) {
    for (int s = 0; s < X_NA; ++s) { mbar_init(&a_full[s], X_CW + 1); mbar_init(&st_done[s], 1); }   // a_full: 16 compute warps + the weight copy
    mbar_init(&acc_full, 1); mbar_init(&acc_empty, X_CW);
    int ns = 0;
    for (int o = 0; o < D::NOUT; ++o) {
      if (D::o_off(o) < 0) continue;
      for (int p = 0; p < D::NPATH; ++p)
        if (D::p_iro(p) == o) { st_o[ns] = (uint8_t)o; st_pidx[ns] = (uint8_t)D::p_pidx(p); ++ns; }
    }
    n_steps_s = ns;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_d0 = tmem_base_s;

  if (warp > X_CW) {
    // ---- weight producers: one bulk copy per (half, path) step; a bulk operation costs its issuing thread ~330 ns, so two
    // threads take alternate steps (X_NW is even: each thread sees every phase of its own slots)
    if (lane == 0) {
      const uint32_t me = warp - (X_CW + 1);
      uint32_t it = 0;
      const int n_steps = n_steps_s;
      XT_DECL
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x)
        for (int half = 0; half < 2; ++half)
          for (int sp = 0; sp < n_steps; ++sp, ++it) {
            if ((it & 1) != me) continue;
            const uint32_t slot = it % X_NW, ph = (it / X_NW) & 1;
            XT(0, x_wait(&st_done[slot], ph ^ 1))
            bulk_g2s(w_ring + (size_t)slot * X_W_BYTES, xa.Bp[st_o[sp]] + (size_t)(2 * st_pidx[sp] + half) * X_W_BYTES, X_W_BYTES, &a_full[slot]);
          }
      if (me == 0) XT_PRINT("producer: w0 = wait w_empty")
    }
  } else if (warp == X_CW) {
    // ---- MMA issuer
    if (lane == 0) {
      // D fp32 (bit 4), A / B format at bits 7 / 10 (0 = fp16, 1 = bf16), K-major, N >> 3 at bit 17, M >> 4 at bit 24
      const uint32_t idesc = (1u << 4) | ((uint32_t)(X_N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
      const uint32_t idesc_bb = idesc | (1u << 7) | (1u << 10);
      uint32_t it = 0, titer = 0;
      const uint64_t d0a = umma_desc(smem_u32(smem), 128, 512), d0b = umma_desc(smem_u32(w_ring), 128, 512);
      const uint32_t d_hi32 = (uint32_t)(d0a >> 32), da_lo32 = (uint32_t)d0a, db_lo32 = (uint32_t)d0b;
      XT_DECL
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++titer) {
        XT(0, x_wait(&acc_empty, (titer & 1) ^ 1))
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int n_steps = n_steps_s;
        for (int half = 0; half < 2; ++half)
          for (int sp = 0; sp < n_steps; ++sp, ++it) {
            const int o = st_o[sp];
            const bool first = half == 0 && (sp == 0 || st_o[sp - 1] != o);
            const uint32_t as = it % X_NA, aph = (it / X_NA) & 1, ws = as;
            XT(1, x_wait(&a_full[as], aph))
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the compute warps' generic-proxy stores (ordered before this
                                                                           // point by the barrier) -> visible to the tensor core
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            // The issuing thread is a single in-order instruction stream: per step it can afford tens of instructions, not
            // hundreds (measured: 808 cycles per step with ten descriptors built from scratch, against 312 of tensor-pipe
            // time).  A descriptor's low word holds the start address (>> 4) and the LBO field, its high word is constant:
            // one add per descriptor.
            const uint32_t fa = da_lo32 + as * (X_A_BYTES >> 4), fb = db_lo32 + ws * (X_W_BYTES >> 4);
            x_step_mma(tmem_d0 + (uint32_t)o * X_N, idesc, idesc_bb, first ? 0u : 1u, d_hi32, fa, fb);
            umma_commit(&st_done[as]);
          }
        umma_commit(&acc_full);
      }
      XT_PRINT("mma: w0 = acc_empty, w1 = a_full, w2 = w_full")
    }
  } else {
    // ---- compute warps.  Warp w: edges 4 (w & 3) + (lane >> 3), channel chunk j = w >> 2 (8 channels), c8 = lane & 7
    const int el = 4 * (warp & 3) + (lane >> 3), j = warp >> 2, c8 = lane & 7;
    const int quad = warp & 3;
    constexpr int n = X_N;
    constexpr int nsc = n * (D::LMAX + 1);
    uint32_t it = 0, titer = 0;
    XT_DECL
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++titer) {
      const int64_t e = tile * X_EDGES + el;
#ifdef X_TRACE
      const unsigned long long tl0 = clock64();
#endif
      const bool valid = e < M;
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        const int c = half * 32 + 8 * j + c8;
        float V[D::IN_DIM], G[D::DSH];
#pragma unroll
        for (int k = 0; k < D::IN_DIM; ++k) V[k] = 0.f;
#pragma unroll
        for (int k = 0; k < D::DSH; ++k) G[k] = 0.f;
        if (valid) {
          if (ly.layer1) {
            float Y[16];
            const float* gp = io.geo + e * GEO_W;
            sph_harm<D::LMAX>(gp[0], gp[1], gp[2], Y);
            const float* wi = io.winit + e * io.ldwi + c;
#pragma unroll
            for (int k = 0; k < D::IN_DIM; ++k) V[k] = wi[l_of_lm(k) * n] * Y[k];   // F5
          } else {
            const float* vp = io.vprev + e * D::IN_DIM * n + c;
#pragma unroll
            for (int k = 0; k < D::IN_DIM; ++k) V[k] = vp[k * n];
          }
          const float* ga = io.gamma + (int64_t)io.e_center[e] * D::DSH * n + c;
#pragma unroll
          for (int k = 0; k < D::DSH; ++k) G[k] = ga[k * n];
        }
#ifdef X_TRACE
        xt[1] += clock64() - tl0;   // (first half only meaningful: load phase)
#endif
#pragma unroll
        for (int o = 0; o < D::NOUT; ++o) {
          const bool lin = D::o_off(o) >= 0;
          if (!lin && o != 0) continue;
          constexpr int dummy = 0; (void)dummy;
          const int d3 = D::o_d3(o);
#pragma unroll
          for (int p = 0; p < D::NPATH; ++p) {
            if (D::p_iro(p) != o) continue;
            float t[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            tpgen::tp_path_fwd<SIG>(p, RegAcc<D::IN_DIM>{V}, RegAcc<D::DSH>{G}, [&](int m, float v) { t[m] = v; });
            if (o == 0 && valid) io.s[e * nsc + D::p_pidx(p) * n + c] = t[0];   // F9
            if (lin) {
              const uint32_t as = it % X_NA, aph = (it / X_NA) & 1;
              XT(0, x_wait(&st_done[as], aph ^ 1))
              uint8_t* ab = smem + (size_t)as * X_A_BYTES;
              // two values per conversion: the packed fp32 -> fp16 / bf16 instructions run on the ALU pipe, the scalar ones at a
              // quarter of its rate (measured: the scalar form made the compute warps the bottleneck)
              const int r0 = el * d3;
#pragma unroll
              for (int m = 0; m < 8; m += 2) {
                if (m >= d3) break;
                const float t1 = (m + 1 < d3) ? t[m + 1 < 7 ? m + 1 : 6] : 0.f;
                const __half2 hi2 = __floats2half2_rn(t[m], t1);
                const float2 hf = __half22float2(hi2);
                const __nv_bfloat162 lo2 = __floats2bfloat162_rn(t[m] - hf.x, t1 - hf.y);
                const uint32_t hb = *reinterpret_cast<const uint32_t*>(&hi2), lb = *reinterpret_cast<const uint32_t*>(&lo2);
                {
                  const int r = r0 + m;
                  const uint32_t off = (uint32_t)(r >> 3) * 512 + j * 128 + (r & 7) * 16 + c8 * 2;
                  *reinterpret_cast<uint16_t*>(ab + off) = (uint16_t)hb;
                  *reinterpret_cast<uint16_t*>(ab + X_A_BYTES / 2 + off) = (uint16_t)lb;
                }
                if (m + 1 < d3) {
                  const int r = r0 + m + 1;
                  const uint32_t off = (uint32_t)(r >> 3) * 512 + j * 128 + (r & 7) * 16 + c8 * 2;
                  *reinterpret_cast<uint16_t*>(ab + off) = (uint16_t)(hb >> 16);
                  *reinterpret_cast<uint16_t*>(ab + X_A_BYTES / 2 + off) = (uint16_t)(lb >> 16);
                }
              }
              __syncwarp();
              if (lane == 0) x_arrive(&a_full[as]);
              ++it;
            }
          }
        }
      }
      // ---- epilogue: TMEM lane r = (edge, m) row of irrep o; this warp reads lanes 32 quad .. + 31 of the irreps o = j, j + 4
      XT(2, x_wait(&acc_full, titer & 1))
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#ifdef X_TRACE
      const unsigned long long te0 = clock64();
#endif
#pragma unroll
      for (int o = 0; o < D::NOUT; ++o) {
        if (D::o_off(o) < 0 || (o & 3) != j) continue;
        const int d3 = D::o_d3(o);
        const int r = quad * 32 + lane;
        const int er = r / d3, mr = r - er * d3;
        const int64_t eo = tile * X_EDGES + er;
        const bool ok = er < X_EDGES && eo < M;
        const float osc = *xa.oscale[o];
        float* dst = io.vout + ((eo * D::OUT_DIM + D::o_off(o) + mr) * n);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          float v[16];
          tmem_ld16(tmem_d0 + ((uint32_t)(quad * 32) << 16) + (uint32_t)(o * X_N + q * 16), v);
          if (ok) {
#pragma unroll
            for (int x = 0; x < 4; ++x)
              *reinterpret_cast<float4*>(dst + q * 16 + 4 * x) = make_float4(v[4 * x] * osc, v[4 * x + 1] * osc, v[4 * x + 2] * osc, v[4 * x + 3] * osc);
          }
        }
      }
#ifdef X_TRACE
      xt[3] += clock64() - te0;
#endif
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) x_arrive(&acc_empty);
    }
    if (tid == 0) XT_PRINT("compute warp 0: w0 = a_empty, w1 = loads(cumulative from tile start), w2 = acc_full, w3 = epilogue")
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d0), "r"(512));
  }
}

template <int SIG>
bool launch_one(Model* m, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, const XArgs& xa) {
  using D = tpgen::SigDims<SIG>;
  if (D::NOUT > 8) return false;
  static int attr_dev = -1;
  if (attr_dev != m->device) {
    if (cudaFuncSetAttribute(k_tpmix_fwd<SIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)X_SMEM) != cudaSuccess) { cudaGetLastError(); return false; }
    attr_dev = m->device;
  }
  k_tpmix_fwd<SIG><<<(unsigned)std::max(1, m->num_sms), X_T, X_SMEM, st>>>(tp, io, xa);
  return true;
}

}  // namespace

// Returns false when the layer is outside what the kernel takes (the caller then uses k_tpo_fwd + one GEMM per irrep).
bool launch_tpmix_fwd(Model* m, int sig, cudaStream_t st, const TpLayerDev& tp, const TpIo& io) {
  if (tp.n != X_N || !tp.has_lin || tp.n_out > TP3_MAXO || !io.vout) return false;
  XArgs xa{};
  for (int o = 0; o < tp.n_out; ++o) {
    if (tp.out_off[o] < 0) continue;
    GemmArgs gm;
    gm.W = io.w + tp.wlin[o]; gm.ldw = tp.out_np[o] * tp.n; gm.wtrans = 0; gm.N = tp.n; gm.K0 = tp.out_np[o] * tp.n; gm.K1 = 0;
    xa.Bp[o] = f16s_packed_weights(m, gm, st, &xa.oscale[o]);
    if (!xa.Bp[o]) return false;
  }
  switch (sig) {
#define X(I) case I: return launch_one<I>(m, st, tp, io, xa);
    TPGEN_FOR_EACH_SIG(X)
#undef X
    default: return false;
  }
}

}  // namespace allegro
