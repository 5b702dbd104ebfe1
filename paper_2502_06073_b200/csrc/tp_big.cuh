// tp_big.cuh — F8/F9 and B5/B8 for networks with many tensor channels (n = 64, 128, 256), where the channel-mixing
// linear W_lin (F11 / B2) is a real GEMM (K = paths x n up to several hundred, N = n) and belongs on tcgen05.
// The tensor product and the mixing are therefore split:
//   forward:   k_tpo_fwd  writes T_o[(e, m)][pidx n + c] per output irrep o (generated coupling code, one (edge, channel)
//              pair per thread, V / Gamma in registers), then gemm_tc.cu forms V^L[e, o, m, :] = T_o W_o^T with the rows
//              mapped straight into the [e][comp][c] layout;
//   backward:  gemm_tc.cu forms Tbar_o = Vbar^L[., o, ., :] W_o per irrep, then k_tpo_bwd applies B5 (+ B4's sbar, + B8
//              for layer 1) with the adjoints in registers.
// T costs d3 x paths x n floats per edge and irrep; the caller sizes its atom chunks for it (network.cu).
// PAPER.md:93 ("64 tensor features ... in full O(3) symmetry"), readings A8, A9, A12; layouts as in tp.cuh.
#pragma once
#include "tc_common.cuh"
#include "tp3.cuh"

namespace allegro {

struct TpBig {
  float* T[TP3_MAXO];      // per output irrep: [E][d3][np n]
};

template <int SIG>
__global__ void __launch_bounds__(256) k_tpo_fwd(TpLayerDev ly, TpIo io, TpBig big) {
  using D = tpgen::SigDims<SIG>;
  const int n = ly.n;
  const DivN divn(n);
  const int64_t M = *io.Mptr;
  const int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x;
  const int64_t e = idx / n;
  const int c = (int)(idx - e * n);
  if (e >= M) return;
  const int nsc = n * (D::LMAX + 1);
  float Y[16], V[D::IN_DIM], G[D::DSH];
  const float* gp = io.geo + e * GEO_W;
  sph_harm<D::LMAX>(gp[0], gp[1], gp[2], Y);
  if (ly.layer1) {
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
#pragma unroll
  for (int p = 0; p < D::NPATH; ++p) {
    const int o = D::p_iro(p), pidx = D::p_pidx(p), d3 = D::o_d3(o);
    const bool lin = ly.has_lin && D::o_off(o) >= 0;
    if (!lin && o != 0) continue;
    const int64_t K = (int64_t)D::o_np(o) * n;
    float* dst = lin ? big.T[o] + (e * d3) * K + pidx * n + c : nullptr;
    float t0 = 0.f;
    tpgen::tp_path_fwd<SIG>(p, RegAcc<D::IN_DIM>{V}, RegAcc<D::DSH>{G}, [&](int m, float v) {
      if (lin) dst[m * K] = v;
      if (m == 0) t0 = v;
    });
    if (o == 0) io.s[e * nsc + pidx * n + c] = t0;   // F9
  }
}

// One block = 256 / n edges x n channels (n a power of two, 64 <= n <= 256).
template <int SIG>
__global__ void __launch_bounds__(256) k_tpo_bwd(TpLayerDev ly, TpIo io, TpBig big) {
  using D = tpgen::SigDims<SIG>;
  __shared__ float ypart[8][16];
  const int n = ly.n;
  const int64_t M = *io.Mptr;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t idx = (int64_t)blockIdx.x * 256 + tid;
  const int64_t e = idx / n;
  const int c = (int)(idx - e * n);
  const bool valid = e < M;
  const int nsc = n * (D::LMAX + 1);
  float Y[16], V[D::IN_DIM], G[D::DSH], Vb[D::IN_DIM], Gb[D::DSH], wil[D::LMAX + 1];
#pragma unroll
  for (int k = 0; k < 16; ++k) Y[k] = 0.f;
#pragma unroll
  for (int k = 0; k < D::IN_DIM; ++k) { V[k] = 0.f; Vb[k] = 0.f; }
#pragma unroll
  for (int k = 0; k < D::DSH; ++k) { G[k] = 0.f; Gb[k] = 0.f; }
#pragma unroll
  for (int l = 0; l <= D::LMAX; ++l) wil[l] = 0.f;
  if (valid) {
    const float* gp = io.geo + e * GEO_W;
    sph_harm<D::LMAX>(gp[0], gp[1], gp[2], Y);
    if (ly.layer1) {
      const float* wi = io.winit + e * io.ldwi + c;
#pragma unroll
      for (int l = 0; l <= D::LMAX; ++l) wil[l] = wi[l * n];
#pragma unroll
      for (int k = 0; k < D::IN_DIM; ++k) V[k] = wil[l_of_lm(k)] * Y[k];
    } else {
      const float* vp = io.vprev + e * D::IN_DIM * n + c;
#pragma unroll
      for (int k = 0; k < D::IN_DIM; ++k) V[k] = vp[k * n];
    }
    const float* ga = io.gamma + (int64_t)io.e_center[e] * D::DSH * n + c;
#pragma unroll
    for (int k = 0; k < D::DSH; ++k) G[k] = ga[k * n];
#pragma unroll
    for (int p = 0; p < D::NPATH; ++p) {
      const int o = D::p_iro(p), pidx = D::p_pidx(p), d3 = D::o_d3(o);
      const bool lin = ly.has_lin && D::o_off(o) >= 0;
      if (!lin && o != 0) continue;
      const int64_t K = (int64_t)D::o_np(o) * n;
      const float* tb = lin ? big.T[o] + (e * d3) * K + pidx * n + c : nullptr;
      const float sb = (o == 0) ? io.sbar[e * nsc + pidx * n + c] : 0.f;
      tpgen::tp_path_bwd<SIG>(p, RegAcc<D::IN_DIM>{V}, RegAcc<D::DSH>{G}, [&](int m) { return (lin ? tb[m * K] : 0.f) + sb; },
                              [&](int k, float v) { Vb[k] += v; }, [&](int k, float v) { Gb[k] += v; });
    }
    float* gout = io.ge + e * D::DSH * n + c;
#pragma unroll
    for (int k = 0; k < D::DSH; ++k) gout[k * n] = Gb[k];
    if (!ly.layer1) {
      float* vo = io.vbar_prev + e * D::IN_DIM * n + c;
#pragma unroll
      for (int k = 0; k < D::IN_DIM; ++k) vo[k * n] = Vb[k];
    }
  }
  if (ly.layer1) {
    // B8: wbar_init[e, l, c] = sum_m Vbar0[lm] Y_lm;  Ybar[e, lm] += sum_c (W_init x0)[l, c] Vbar0[lm, c]
    if (valid) {
#pragma unroll
      for (int l = 0; l <= D::LMAX; ++l) {
        float sacc = 0.f;
#pragma unroll
        for (int mm = 0; mm < 2 * l + 1; ++mm) sacc = fmaf(Vb[l * l + mm], Y[l * l + mm], sacc);
        io.wbar_init[e * io.ldwb + l * n + c] = sacc;
      }
    }
    if constexpr (D::IN_DIM == D::DSH) {
      // channels of one edge span n / 32 whole warps: warp sums by shuffle, then a fixed-order sum of the warp partials
      const int wpe = n >> 5;
#pragma unroll
      for (int k = 0; k < D::DSH; ++k) {
        float v = wil[l_of_lm(k)] * Vb[k];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        if (lane == 0) ypart[warp][k] = v;
      }
      __syncthreads();
      if ((warp % wpe) == 0 && lane < D::DSH && valid) {
        float s = 0.f;
        for (int w2 = 0; w2 < wpe; ++w2) s += ypart[warp + w2][lane];
        io.ybar[e * D::DSH + lane] += s;
      }
    }
  }
}

// ---- k_tpo_bwd_ring: k_tpo_bwd with the T-bar values staged through shared memory by bulk copies.
// k_tpo_bwd reads one T-bar value per coupling term per thread straight from HBM and is bound by the latency of those loads
// (37 % of the DRAM peak at 24 % of the warp slots, profiles/r2_d_launches_cfg3.md): the bytes in flight are limited by the
// registers that wait for them.  Here one persistent CTA per SM walks groups of 256 / n edges; a producer thread copies the
// T-bar block of (group, output irrep) — contiguous in T_o[E][d3][np n] — into a ring of shared-memory slots with one
// cp.async.bulk each (tens of KB in flight per SM whatever the register count), and the 256 compute threads (one (edge, channel)
// pair each, adjoints in registers as before) take the paths irrep by irrep from the slot.  Same arithmetic per path; the paths
// are visited in irrep order, so the fp32 sums of Vbar / Gbar differ from k_tpo_bwd in rounding order only.
template <int SIG>
struct TpoRing {
  using D = tpgen::SigDims<SIG>;
  static constexpr int max_units() {
    int mx = 1;
    for (int o = 0; o < D::NOUT; ++o)
      if (D::o_off(o) >= 0 && D::o_d3(o) * D::o_np(o) > mx) mx = D::o_d3(o) * D::o_np(o);
    return mx;
  }
  static constexpr uint32_t SLOT = (uint32_t)max_units() * 1024u;   // 256 (edge, channel) pairs x 4 bytes per (m, path)
};
constexpr int TPO_RING_T = 288;                                     // 8 compute warps + 1 producer warp
constexpr int TPO_RING_MAX_SLOTS = 4;

__device__ __forceinline__ void tpo_wait(uint64_t* bar, uint32_t parity) {   // bounded: a protocol error traps instead of hanging
  uint32_t done = 0;
  for (uint32_t it = 0; !done; ++it) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity), "r"(1000u)
        : "memory");
    if (it > (1u << 22)) __trap();
  }
}

template <int SIG>
__global__ void __launch_bounds__(TPO_RING_T, 1) k_tpo_bwd_ring(TpLayerDev ly, TpIo io, TpBig big, int n_slots) {
  using D = tpgen::SigDims<SIG>;
  extern __shared__ uint8_t tpo_smem_dyn[];
  __shared__ __align__(8) uint64_t full[TPO_RING_MAX_SLOTS], empty[TPO_RING_MAX_SLOTS];
  __shared__ float ypart[8][16];
  uint8_t* ring = tpo_smem_dyn + ((128u - (smem_u32(tpo_smem_dyn) & 127u)) & 127u);
  const int n = ly.n;
  const int EG = 256 / n;                                           // edges per group
  const int64_t M = *io.Mptr;
  const int64_t n_groups = (M + EG - 1) / EG;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid == 0) {
    for (int s = 0; s < n_slots; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (warp == 8) {
    // ---- producer
    if (lane == 0) {
      uint32_t it = 0;
      for (int64_t g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const int64_t e0 = g * EG;
        const int64_t ne = (M - e0 < EG) ? (M - e0) : EG;
#pragma unroll
        for (int o = 0; o < D::NOUT; ++o) {
          if (!(ly.has_lin && D::o_off(o) >= 0)) continue;
          const uint32_t slot = it % (uint32_t)n_slots, ph = (it / (uint32_t)n_slots) & 1;
          tpo_wait(&empty[slot], ph ^ 1);
          const int64_t K = (int64_t)D::o_np(o) * n;
          bulk_g2s(ring + (size_t)slot * TpoRing<SIG>::SLOT, big.T[o] + e0 * D::o_d3(o) * K, (uint32_t)(ne * D::o_d3(o) * K * 4), &full[slot]);
          ++it;
        }
      }
    }
    return;
  }
  // ---- compute: thread = (edge of the group, channel)
  const int el = tid / n, c = tid - el * n;
  const int nsc = n * (D::LMAX + 1);
  uint32_t it = 0;
  for (int64_t g = blockIdx.x; g < n_groups; g += gridDim.x) {
    const int64_t e = g * EG + el;
    const bool valid = e < M;
    float Y[16], V[D::IN_DIM], G[D::DSH], Vb[D::IN_DIM], Gb[D::DSH], wil[D::LMAX + 1];
#pragma unroll
    for (int k = 0; k < 16; ++k) Y[k] = 0.f;
#pragma unroll
    for (int k = 0; k < D::IN_DIM; ++k) { V[k] = 0.f; Vb[k] = 0.f; }
#pragma unroll
    for (int k = 0; k < D::DSH; ++k) { G[k] = 0.f; Gb[k] = 0.f; }
#pragma unroll
    for (int l = 0; l <= D::LMAX; ++l) wil[l] = 0.f;
    if (valid) {
      const float* gp = io.geo + e * GEO_W;
      sph_harm<D::LMAX>(gp[0], gp[1], gp[2], Y);
      if (ly.layer1) {
        const float* wi = io.winit + e * io.ldwi + c;
#pragma unroll
        for (int l = 0; l <= D::LMAX; ++l) wil[l] = wi[l * n];
#pragma unroll
        for (int k = 0; k < D::IN_DIM; ++k) V[k] = wil[l_of_lm(k)] * Y[k];
      } else {
        const float* vp = io.vprev + e * D::IN_DIM * n + c;
#pragma unroll
        for (int k = 0; k < D::IN_DIM; ++k) V[k] = vp[k * n];
      }
      const float* ga = io.gamma + (int64_t)io.e_center[e] * D::DSH * n + c;
#pragma unroll
      for (int k = 0; k < D::DSH; ++k) G[k] = ga[k * n];
    }
#pragma unroll
    for (int o = 0; o < D::NOUT; ++o) {
      const bool lin = ly.has_lin && D::o_off(o) >= 0;
      if (!lin && o != 0) continue;
      const int d3 = D::o_d3(o);
      const int K = D::o_np(o) * n;
      uint32_t slot = 0;
      if (lin) {
        slot = it % (uint32_t)n_slots;
        tpo_wait(&full[slot], (it / (uint32_t)n_slots) & 1);
      }
      if (valid) {
        const float* tslot = reinterpret_cast<const float*>(ring + (size_t)slot * TpoRing<SIG>::SLOT) + (el * d3) * K + c;
#pragma unroll
        for (int p = 0; p < D::NPATH; ++p) {
          if (D::p_iro(p) != o) continue;
          const int pidx = D::p_pidx(p);
          const float* tb = tslot + pidx * n;
          const float sb = (o == 0) ? io.sbar[e * nsc + pidx * n + c] : 0.f;
          tpgen::tp_path_bwd<SIG>(p, RegAcc<D::IN_DIM>{V}, RegAcc<D::DSH>{G}, [&](int m) { return (lin ? tb[m * K] : 0.f) + sb; },
                                  [&](int k, float v) { Vb[k] += v; }, [&](int k, float v) { Gb[k] += v; });
        }
      }
      if (lin) {
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&empty[slot])) : "memory");
        ++it;
      }
    }
    if (valid) {
      float* gout = io.ge + e * D::DSH * n + c;
#pragma unroll
      for (int k = 0; k < D::DSH; ++k) gout[k * n] = Gb[k];
      if (!ly.layer1) {
        float* vo = io.vbar_prev + e * D::IN_DIM * n + c;
#pragma unroll
        for (int k = 0; k < D::IN_DIM; ++k) vo[k * n] = Vb[k];
      }
    }
    if (ly.layer1) {
      // B8 as in k_tpo_bwd
      if (valid) {
#pragma unroll
        for (int l = 0; l <= D::LMAX; ++l) {
          float sacc = 0.f;
#pragma unroll
          for (int mm = 0; mm < 2 * l + 1; ++mm) sacc = fmaf(Vb[l * l + mm], Y[l * l + mm], sacc);
          io.wbar_init[e * io.ldwb + l * n + c] = sacc;
        }
      }
      if constexpr (D::IN_DIM == D::DSH) {
        const int wpe = n >> 5;
        asm volatile("bar.sync 1, 256;" ::: "memory");              // the previous group's ypart has been read
#pragma unroll
        for (int k = 0; k < D::DSH; ++k) {
          float v = wil[l_of_lm(k)] * Vb[k];
#pragma unroll
          for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
          if (lane == 0) ypart[warp][k] = v;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if ((warp % wpe) == 0 && lane < D::DSH && valid) {
          float s = 0.f;
          for (int w2 = 0; w2 < wpe; ++w2) s += ypart[warp + w2][lane];
          io.ybar[e * D::DSH + lane] += s;
        }
      }
    }
  }
}

}  // namespace allegro
