// tp3.cuh — F8/F9/F11 and B2/B5/B8 for networks with few tensor channels (n in {8, 16, 32}): persistent blocks, one
// (edge, channel) pair per thread with V, Gamma (and, backward, their adjoints) in registers, the generated coupling
// code of tp_gen.cuh fully unrolled over the layer's paths, and the channel-mixing linear W_lin on the tensor cores
// (warp-level mma.sync m16n8k8 TF32 with the 3-pass hi/lo split: same error class as fp32 FMA, see gemm_tc.cu).
// W_lin (hi/lo split) stays in shared memory for the whole life of the block.
// PAPER.md:93 ("tensor features with l=2 in full O(3) symmetry"), readings A8, A9, A12; layouts as in tp.cuh.
#pragma once
#include "tp.cuh"

namespace allegro {

__device__ __forceinline__ uint32_t tf32_hi(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void mma_tf32(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

constexpr int TP3_MAXO = 8;
struct Tp3Smem {            // per-irrep tile geometry, filled by thread 0
  int lin[TP3_MAXO], K[TP3_MAXO], ldk[TP3_MAXO], d3[TP3_MAXO], ooff[TP3_MAXO], boff[TP3_MAXO], toff[TP3_MAXO], aoff[TP3_MAXO],
      unit0[TP3_MAXO + 1];
};

// shared-memory floats needed by the v3 kernels (host and device use the same formula)
__host__ __device__ inline int tp3_round16(int x) { return (x + 15) / 16 * 16; }

// register-array accessors for the generated code
template <int N> struct RegAcc {
  const float (&r)[N];
  __device__ __forceinline__ float operator()(int k) const { return r[k]; }
};

// One unit of the channel-mixing GEMM: 16 rows x (8 NB) output channels, K deep, 3-pass TF32 (hi/lo) with the A fragments
// split on the fly and the pre-split B fragments read from shared memory (lo block at offset lo_off).  NB = n / 8.
template <int NB>
__device__ __forceinline__ void tp3_fwd_unit(const float* __restrict__ Ta, int ldk, const float* __restrict__ Bh, int lo_off, int ldn,
                                             int K, int row_g, int d3, int TE, int64_t e0, int64_t M, float* __restrict__ out0,
                                             int edge_stride, int n) {
  float acc[NB][4];
#pragma unroll
  for (int nb = 0; nb < NB; ++nb)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[nb][j] = 0.f;
  const float* ta = Ta;
  const float* bh = Bh;
  const int ldk8 = 8 * ldk, ldn4 = 4 * ldn, ldn8 = 8 * ldn;
  for (int k0 = 0; k0 < K; k0 += 8) {
    const float a[4] = {ta[0], ta[ldk8], ta[4], ta[ldk8 + 4]};
    uint32_t ah[4], al[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { ah[j] = tf32_hi(a[j]); al[j] = __float_as_uint(a[j] - __uint_as_float(ah[j])); }
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) {
      const uint32_t b0h = __float_as_uint(bh[nb * 8]), b1h = __float_as_uint(bh[ldn4 + nb * 8]);
      const uint32_t b0l = __float_as_uint(bh[lo_off + nb * 8]), b1l = __float_as_uint(bh[lo_off + ldn4 + nb * 8]);
      mma_tf32(acc[nb], al, b0h, b1h);
      mma_tf32(acc[nb], ah, b0l, b1l);
      mma_tf32(acc[nb], ah, b0h, b1h);
    }
    ta += 8; bh += ldn8;
  }
  const DivS divd3(d3);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    int e2, m;
    divd3(row_g + 8 * h, &e2, &m);
    if (e2 < TE && e0 + e2 < M) {
      float* out = out0 + (e0 + e2) * edge_stride + m * n;
#pragma unroll
      for (int nb = 0; nb < NB; ++nb) *reinterpret_cast<float2*>(out + nb * 8) = make_float2(acc[nb][2 * h], acc[nb][2 * h + 1]);
    }
  }
}

// Backward unit: Tb[16 rows, K_o] = A[16 rows, n] B[n, K_o]; the A fragments of the KS = n / 8 k-steps are split once.
template <int KS>
__device__ __forceinline__ void tp3_bwd_unit(const float* __restrict__ A, int lda, const float* __restrict__ Bh, int lo_off, int ldb,
                                             int K, float* __restrict__ Tb, int ldk) {
  uint32_t ah[KS][4], al[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    const float a[4] = {A[ks * 8], A[ks * 8 + 8 * lda], A[ks * 8 + 4], A[ks * 8 + 8 * lda + 4]};
#pragma unroll
    for (int j = 0; j < 4; ++j) { ah[ks][j] = tf32_hi(a[j]); al[ks][j] = __float_as_uint(a[j] - __uint_as_float(ah[ks][j])); }
  }
  const int ldb4 = 4 * ldb, ldb8 = 8 * ldb, ldk8 = 8 * ldk;
  for (int nb8 = 0; nb8 < K; nb8 += 8) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    const float* bh = Bh + nb8;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      const uint32_t b0h = __float_as_uint(bh[0]), b1h = __float_as_uint(bh[ldb4]);
      const uint32_t b0l = __float_as_uint(bh[lo_off]), b1l = __float_as_uint(bh[lo_off + ldb4]);
      mma_tf32(acc, al[ks], b0h, b1h);
      mma_tf32(acc, ah[ks], b0l, b1l);
      mma_tf32(acc, ah[ks], b0h, b1h);
      bh += ldb8;
    }
    *reinterpret_cast<float2*>(Tb + nb8) = make_float2(acc[0], acc[1]);
    *reinterpret_cast<float2*>(Tb + ldk8 + nb8) = make_float2(acc[2], acc[3]);
  }
}

// ---------------------------------------------------------------------------------------------------------
// forward.  smem (floats): per mixed irrep o: Bhi[K_o][n+8] | Blo[K_o][n+8]  (B[k][c'] = W_o[c'][k], k = pidx n + c),
// then per mixed irrep o: T_o[rows_o][K_o+4], rows_o = roundup(TE d3_o, 16), row = el d3 + m.
// ---------------------------------------------------------------------------------------------------------
// NCH = number of channels as a compile-time constant (8, 16, 32: strides become immediates, the kernels are issue-bound
// and half of their instructions were address arithmetic), or 0 = read it from the layer descriptor.
template <int SIG, int NCH>
__global__ void __launch_bounds__(256, 3) k_tp_fwd3(TpLayerDev ly, TpIo io) {
  using D = tpgen::SigDims<SIG>;
  extern __shared__ __align__(16) float sm[];
  __shared__ Tp3Smem g;
  const int n = NCH ? NCH : ly.n, ldn = n + 8;
  const DivN divn(n);
  const int TE = 256 / n;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, gq = lane >> 2, tq = lane & 3;
  int el, c;
  divn(tid, &el, &c);
  const int64_t M = *io.Mptr;
  const int64_t nsub = (M + TE - 1) / TE;
  if ((int64_t)blockIdx.x >= nsub) return;
  const int nsc = n * (D::LMAX + 1);
  if (tid == 0) {
    int off = 0, units = 0;
    for (int o = 0; o < D::NOUT; ++o) {
      g.lin[o] = (ly.has_lin && D::o_off(o) >= 0) ? 1 : 0;
      g.K[o] = D::o_np(o) * n; g.ldk[o] = g.K[o] + 4; g.d3[o] = D::o_d3(o); g.ooff[o] = D::o_off(o);
      g.boff[o] = off;
      if (g.lin[o]) off += 2 * g.K[o] * ldn;
    }
    for (int o = 0; o < D::NOUT; ++o) {
      g.toff[o] = off; g.unit0[o] = units;
      if (g.lin[o]) { const int rows = tp3_round16(TE * g.d3[o]); off += rows * g.ldk[o]; units += rows / 16; }
    }
    g.unit0[D::NOUT] = units;
  }
  __syncthreads();
  // W_lin -> shared memory once per block, split hi/lo
  for (int o = 0; o < D::NOUT; ++o) {
    if (!g.lin[o]) continue;
    const float* Wo = io.w + ly.wlin[o];
    const int K = g.K[o];
    float* Bh = sm + g.boff[o];
    float* Bl = Bh + K * ldn;
    for (int idx = tid; idx < K * n; idx += 256) {
      const int cp = idx / K, k = idx - cp * K;
      const float v = Wo[idx];
      const float hi = __uint_as_float(tf32_hi(v));
      Bh[k * ldn + cp] = hi; Bl[k * ldn + cp] = v - hi;
    }
  }
  // this thread's slot in every T tile (irrep index is a compile-time constant in the unrolled path loop below)
  float* tdst[D::NOUT];
  int tld[D::NOUT];
#pragma unroll
  for (int o = 0; o < D::NOUT; ++o) { tld[o] = g.ldk[o]; tdst[o] = sm + g.toff[o] + (el * D::o_d3(o)) * g.ldk[o] + c; }
  for (int64_t st = blockIdx.x; st < nsub; st += gridDim.x) {
    const int64_t e0 = st * TE, e = e0 + el;
    __syncthreads();   // previous sub-tile's T fully consumed (and, first time, W_lin staged)
    if (e < M && el < TE) {
      float Y[16], V[D::IN_DIM], G[D::DSH];
      const float* gp = io.geo + e * GEO_W;
      sph_harm<D::LMAX>(gp[0], gp[1], gp[2], Y);
      if (ly.layer1) {
        const float* wi = io.winit + e * io.ldwi + c;
#pragma unroll
        for (int k = 0; k < D::IN_DIM; ++k) V[k] = wi[l_of_lm(k) * n] * Y[k];   // F5 (IN_DIM == DSH for layer 1)
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
        constexpr int dummy = 0; (void)dummy;
        const int o = D::p_iro(p), pidx = D::p_pidx(p), d3 = D::o_d3(o);
        const bool lin = ly.has_lin && D::o_off(o) >= 0;
        if (!lin && o != 0) continue;
        float* dst = tdst[o] + pidx * n;
        const int ldk = tld[o];
        (void)d3;
        float t0 = 0.f;
        tpgen::tp_path_fwd<SIG>(p, RegAcc<D::IN_DIM>{V}, RegAcc<D::DSH>{G}, [&](int m, float v) {
          if (lin) dst[m * ldk] = v;
          if (m == 0) t0 = v;
        });
        if (o == 0) io.s[e * nsc + pidx * n + c] = t0;   // F9: path-major, then channel
      }
    }
    if (!ly.has_lin) continue;
    __syncthreads();
    // F11 on the tensor cores: unit = 16 rows of one irrep x all n output channels
    const int nunits = g.unit0[D::NOUT];
    for (int u = warp; u < nunits; u += 8) {
      int o = 0;
      while (u >= g.unit0[o + 1]) ++o;
      const int r0 = (u - g.unit0[o]) * 16, K = g.K[o], ldk = g.ldk[o], d3 = g.d3[o];
      const float* Ta = sm + g.toff[o] + (r0 + gq) * ldk + tq;
      const float* Bh = sm + g.boff[o] + tq * ldn + gq;
      float* out0 = io.vout + g.ooff[o] * n + 2 * tq;
      switch (n >> 3) {
        case 1: tp3_fwd_unit<1>(Ta, ldk, Bh, K * ldn, ldn, K, r0 + gq, d3, TE, e0, M, out0, D::OUT_DIM * n, n); break;
        case 2: tp3_fwd_unit<2>(Ta, ldk, Bh, K * ldn, ldn, K, r0 + gq, d3, TE, e0, M, out0, D::OUT_DIM * n, n); break;
        default: tp3_fwd_unit<4>(Ta, ldk, Bh, K * ldn, ldn, K, r0 + gq, d3, TE, e0, M, out0, D::OUT_DIM * n, n); break;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// backward.  smem (floats): per mixed irrep o: Bhi[n][K_o+8] | Blo[n][K_o+8]  (B[c'][col] = W_o[c'][col], col = pidx n + c),
// then per mixed irrep o: A_o[rows_o][n+4] (adjoint of V^L, row = el d3 + m) | Tb_o[rows_o][K_o+4] (adjoint of T).
// Layer 1 applies B8 in registers (wbar_init, Ybar) and never writes Vbar^0.
// ---------------------------------------------------------------------------------------------------------
template <int SIG, int NCH>
__global__ void __launch_bounds__(256, 3) k_tp_bwd3(TpLayerDev ly, TpIo io) {
  using D = tpgen::SigDims<SIG>;
  extern __shared__ __align__(16) float sm[];
  __shared__ Tp3Smem g;
  const int n = NCH ? NCH : ly.n, lda = n + 4;
  const DivN divn(n);
  const int TE = 256 / n;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, gq = lane >> 2, tq = lane & 3;
  int el, c;
  divn(tid, &el, &c);
  const int64_t M = *io.Mptr;
  const int64_t nsub = (M + TE - 1) / TE;
  if ((int64_t)blockIdx.x >= nsub) return;
  const int nsc = n * (D::LMAX + 1);
  if (tid == 0) {
    int off = 0, units = 0;
    for (int o = 0; o < D::NOUT; ++o) {
      g.lin[o] = (ly.has_lin && D::o_off(o) >= 0) ? 1 : 0;
      g.K[o] = D::o_np(o) * n; g.ldk[o] = g.K[o] + 4; g.d3[o] = D::o_d3(o); g.ooff[o] = D::o_off(o);
      g.boff[o] = off;
      if (g.lin[o]) off += 2 * n * (g.K[o] + 8);
    }
    for (int o = 0; o < D::NOUT; ++o) {
      g.unit0[o] = units;
      const int rows = tp3_round16(TE * g.d3[o]);
      g.aoff[o] = off;
      if (g.lin[o]) off += rows * lda;
      g.toff[o] = off;
      if (g.lin[o]) { off += rows * g.ldk[o]; units += rows / 16; }
    }
    g.unit0[D::NOUT] = units;
  }
  __syncthreads();
  for (int o = 0; o < D::NOUT; ++o) {
    if (!g.lin[o]) continue;
    const float* Wo = io.w + ly.wlin[o];
    const int K = g.K[o], ldb = K + 8;
    float* Bh = sm + g.boff[o];
    float* Bl = Bh + n * ldb;
    for (int idx = tid; idx < K * n; idx += 256) {
      const int cp = idx / K, col = idx - cp * K;
      const float v = Wo[idx];
      const float hi = __uint_as_float(tf32_hi(v));
      Bh[cp * ldb + col] = hi; Bl[cp * ldb + col] = v - hi;
    }
  }
  const float* tsrc[D::NOUT];
  float* adst[D::NOUT];
  int tld[D::NOUT];
#pragma unroll
  for (int o = 0; o < D::NOUT; ++o) {
    tld[o] = g.ldk[o];
    tsrc[o] = sm + g.toff[o] + (el * D::o_d3(o)) * g.ldk[o] + c;
    adst[o] = sm + g.aoff[o] + (el * D::o_d3(o)) * lda + c;
  }
  for (int64_t st = blockIdx.x; st < nsub; st += gridDim.x) {
    const int64_t e0 = st * TE, e = e0 + el;
    const bool valid = e < M;
    __syncthreads();
    if (ly.has_lin) {
      // adjoint of V^L for the sub-tile -> A tiles
#pragma unroll
      for (int o = 0; o < D::NOUT; ++o) {
        if (D::o_off(o) < 0) continue;
        float* A = adst[o];
#pragma unroll
        for (int m = 0; m < D::o_d3(o); ++m)
          A[m * lda] = valid ? io.vbar[(e * D::OUT_DIM + D::o_off(o) + m) * n + c] : 0.f;
      }
      __syncthreads();
      // B2 on the tensor cores: Tb_o[rows, K_o] = A_o[rows, n] W_o[n, K_o]
      const int nunits = g.unit0[D::NOUT];
      for (int u = warp; u < nunits; u += 8) {
        int o = 0;
        while (u >= g.unit0[o + 1]) ++o;
        const int r0 = (u - g.unit0[o]) * 16, K = g.K[o], ldk = g.ldk[o], ldb = K + 8;
        const float* A = sm + g.aoff[o] + (r0 + gq) * lda + tq;
        const float* Bh = sm + g.boff[o] + tq * ldb + gq;
        float* Tb = sm + g.toff[o] + (r0 + gq) * ldk + 2 * tq;
        switch (n >> 3) {
          case 1: tp3_bwd_unit<1>(A, lda, Bh, n * ldb, ldb, K, Tb, ldk); break;
          case 2: tp3_bwd_unit<2>(A, lda, Bh, n * ldb, ldb, K, Tb, ldk); break;
          default: tp3_bwd_unit<4>(A, lda, Bh, n * ldb, ldb, K, Tb, ldk); break;
        }
      }
      __syncthreads();
    }
    // B5 (+ B4's sbar, + B8 for layer 1) per (edge, channel) pair, everything in registers
    float Y[16], V[D::IN_DIM], G[D::DSH], Vb[D::IN_DIM], Gb[D::DSH];
#pragma unroll
    for (int k = 0; k < 16; ++k) Y[k] = 0.f;
#pragma unroll
    for (int k = 0; k < D::IN_DIM; ++k) { V[k] = 0.f; Vb[k] = 0.f; }
#pragma unroll
    for (int k = 0; k < D::DSH; ++k) { G[k] = 0.f; Gb[k] = 0.f; }
    float wil[D::LMAX + 1];
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
        const float* tb = tsrc[o] + pidx * n;
        const int ldk = tld[o];
        (void)d3;
        const float sb = (o == 0) ? io.sbar[e * nsc + pidx * n + c] : 0.f;
        tpgen::tp_path_bwd<SIG>(p, RegAcc<D::IN_DIM>{V}, RegAcc<D::DSH>{G},
                                [&](int m) { return (lin ? tb[m * ldk] : 0.f) + sb; },
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
#pragma unroll
        for (int k = 0; k < D::DSH; ++k) {
          float v = wil[l_of_lm(k)] * Vb[k];
          for (int d = n >> 1; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
          if (c == 0 && valid) io.ybar[e * D::DSH + k] += v;
        }
      }
    }
  }
}

}  // namespace allegro
