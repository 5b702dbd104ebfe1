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

}  // namespace allegro
