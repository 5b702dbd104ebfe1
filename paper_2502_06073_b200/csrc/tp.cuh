// tp.cuh — F8/F9/F11 and B2/B5: the channel-wise Clebsch-Gordan tensor product V (x) Gamma of one layer, fused
// with the channel-mixing linear W_lin (forward) / its transpose (backward), so that the per-path product T is
// only ever held as a shared-memory tile ("64 tensor features with l=2 in full O(3) symmetry";
// readings A8, A9, A12).  The sparse coupling tables (nonzeros grouped by output component) live in global
// memory and are read through L1 by every thread in lock-step (uniform control flow).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "device_math.cuh"
#include "model.h"

namespace allegro {

constexpr int TP_MAX_OUT = 8;
constexpr int TP_T = 256;

struct TpLayerDev {
  int n, lmax, dsh, in_dim, out_dim, n_paths, n_out, layer1, has_lin;
  const int* path_tab;     // [n_paths][8]: in_off, d1, l2off, d2, iro, pidx, cg_begin, cg_end
  const int* cg_idx;       // m1 | m2<<8 | m3<<16
  const float* cg_val;
  int out_d3[TP_MAX_OUT], out_off[TP_MAX_OUT], out_np[TP_MAX_OUT];
  long long wlin[TP_MAX_OUT];   // blob offsets of W_lin^{(l,p)}  [n, np*n]
};

struct TpIo {
  const int64_t* Mptr;
  const int* e_center;
  const float* geo;
  const float* gamma;      // [atoms, n, dsh]
  const float* vprev;      // [E, n, in_dim]      (layers >= 2)
  const float* winit; int ldwi;   // [E, .] first n_sc columns = W_init x0   (layer 1)
  const float* w;          // weight blob
  float* s;                // [E, n_sc]   scalars (forward)
  float* vout;             // [E, n, out_dim]     (forward, has_lin)
  // backward
  const float* sbar;       // [E, n_sc]
  const float* vbar;       // [E, n, out_dim]  adjoint of V^L (has_lin)
  float* vbar_prev;        // [E, n, in_dim]
  float* ge;               // [E, n, dsh]  per-edge contribution to Gammabar
};

// value of V^{L-1}[e, c, in_off + m1]
__device__ __forceinline__ float tp_load_v(const TpLayerDev& ly, const TpIo& io, int64_t e, int c, int in_off, int d1, int m1,
                                           const float* Ys_e) {
  if (ly.layer1) {
    const int l1 = (d1 - 1) >> 1;
    return io.winit[e * io.ldwi + c * (ly.lmax + 1) + l1] * Ys_e[in_off + m1];   // V^0 = (W_init x0)_{c,l} Y_lm (F5); in_off = l^2
  }
  return io.vprev[(e * ly.n + c) * ly.in_dim + in_off + m1];
}

// ---------------------------------------------------------------------------------------------------------
// forward: grid = (edge tiles, out irreps).  smem: Tt[n][R] | Ws[n][n] | Ys[TE][16]
// ---------------------------------------------------------------------------------------------------------
constexpr int TP_MAXMT = 4;   // 4x4 micro-tiles per thread

__global__ void __launch_bounds__(TP_T) k_tp_fwd(TpLayerDev ly, TpIo io, int TE) {
  extern __shared__ __align__(16) float sm[];
  const int64_t M = *io.Mptr;
  const int64_t e0 = (int64_t)blockIdx.x * TE;
  if (e0 >= M) return;
  const int o = blockIdx.y;
  const int n = ly.n, d3 = ly.out_d3[o];
  const int R = TE * d3;                       // TE is a multiple of 4
  float* Tt = sm;                              // [n][R]
  float* Ws = Tt + n * R;                      // [n][n]  Ws[c][c'] = W[c', pidx n + c]
  float* Ys = Ws + n * n;                      // [TE][16]
  const int tid = threadIdx.x;
  const int ne = (int)min((int64_t)TE, M - e0);
  for (int t = tid; t < TE; t += TP_T) {
    float* y = Ys + t * 16;
    if (t < ne) { const float* gq = io.geo + (e0 + t) * GEO_W; sph_harm_rt(ly.lmax, gq[0], gq[1], gq[2], y); }
  }
  const bool lin = ly.has_lin && ly.out_off[o] >= 0;
  const int ntr = R >> 2, ntc = n >> 2, nmt = ntr * ntc;
  float acc[TP_MAXMT][4][4];
#pragma unroll
  for (int q = 0; q < TP_MAXMT; ++q)
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[q][i][j] = 0.f;
  const float* Wo = lin ? io.w + ly.wlin[o] : nullptr;
  const int ldw = ly.out_np[o] * n;
  __syncthreads();
  for (int p = 0; p < ly.n_paths; ++p) {
    const int* pt = ly.path_tab + p * 8;
    if (pt[4] != o) continue;
    const int in_off = pt[0], d1 = pt[1], l2off = pt[2], pidx = pt[5], cb = pt[6], ce = pt[7];
    // T_p[e, c, m3] for the tile
    for (int idx = tid; idx < TE * n; idx += TP_T) {
      const int el = idx % TE, c = idx / TE;
      float* dst = Tt + c * R + el * d3;
      if (el >= ne) { for (int m = 0; m < d3; ++m) dst[m] = 0.f; continue; }
      const int64_t e = e0 + el;
      const float* G = io.gamma + ((int64_t)io.e_center[e] * n + c) * ly.dsh + l2off;
      const float* Ye = Ys + el * 16;
      float a = 0.f; int cur = -1;
      for (int m = 0; m < d3; ++m) dst[m] = 0.f;
      for (int q = cb; q < ce; ++q) {
        const int pk = ly.cg_idx[q];
        const int m1 = pk & 255, m2 = (pk >> 8) & 255, m3 = pk >> 16;
        if (m3 != cur) { if (cur >= 0) dst[cur] = a; cur = m3; a = 0.f; }
        a = fmaf(ly.cg_val[q] * tp_load_v(ly, io, e, c, in_off, d1, m1, Ye), G[m2], a);
      }
      if (cur >= 0) dst[cur] = a;
      if (o == 0) io.s[e * (n * (ly.lmax + 1)) + pidx * n + c] = dst[0];   // F9: path-major, then channel
    }
    if (lin) {
      for (int idx = tid; idx < n * n; idx += TP_T) {
        const int cp = idx / n, c = idx - cp * n;           // coalesced along c
        Ws[c * n + cp] = Wo[(int64_t)cp * ldw + pidx * n + c];
      }
    }
    __syncthreads();
    if (lin) {
#pragma unroll
      for (int q = 0; q < TP_MAXMT; ++q) {
        const int mt = tid + q * TP_T;
        if (mt < nmt) {
          const int tr = mt % ntr, tc = mt / ntr;
          for (int k = 0; k < n; ++k) {
            const float4 av = *reinterpret_cast<const float4*>(Tt + k * R + tr * 4);
            const float4 bv = *reinterpret_cast<const float4*>(Ws + k * n + tc * 4);
            const float a4[4] = {av.x, av.y, av.z, av.w}, b4[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int j = 0; j < 4; ++j) acc[q][i][j] = fmaf(a4[i], b4[j], acc[q][i][j]);
          }
        }
      }
    }
    __syncthreads();
  }
  if (lin) {
    const int ooff = ly.out_off[o];
#pragma unroll
    for (int q = 0; q < TP_MAXMT; ++q) {
      const int mt = tid + q * TP_T;
      if (mt < nmt) {
        const int tr = mt % ntr, tc = mt / ntr;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int r = tr * 4 + i, el = r / d3, m = r - el * d3;
          if (el < ne) {
#pragma unroll
            for (int j = 0; j < 4; ++j) io.vout[((e0 + el) * n + tc * 4 + j) * ly.out_dim + ooff + m] = acc[q][i][j];
          }
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// backward: one block per TE edges, all out irreps and paths.
// smem: VB[TE][n][in_dim] | GE[TE][n][dsh] | At[n][Rmax] | Tt[n][Rmax] | Ws[n][n] | Ys[TE][16]
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TP_T) k_tp_bwd(TpLayerDev ly, TpIo io, int TE, int d3max) {
  extern __shared__ __align__(16) float sm[];
  const int64_t M = *io.Mptr;
  const int64_t e0 = (int64_t)blockIdx.x * TE;
  if (e0 >= M) return;
  const int n = ly.n, Rmax = TE * d3max;
  float* VB = sm;
  float* GE = VB + TE * n * ly.in_dim;
  float* At = GE + TE * n * ly.dsh;
  float* Tt = At + n * Rmax;
  float* Ws = Tt + n * Rmax;
  float* Ys = Ws + n * n;
  const int tid = threadIdx.x;
  const int ne = (int)min((int64_t)TE, M - e0);
  for (int t = tid; t < TE; t += TP_T)
    if (t < ne) { const float* gq = io.geo + (e0 + t) * GEO_W; sph_harm_rt(ly.lmax, gq[0], gq[1], gq[2], Ys + t * 16); }
  for (int idx = tid; idx < TE * n * (ly.in_dim + ly.dsh); idx += TP_T) VB[idx] = 0.f;   // VB and GE are adjacent
  __syncthreads();
  for (int o = 0; o < ly.n_out; ++o) {
    const int d3 = ly.out_d3[o], R = TE * d3;
    const bool lin = ly.has_lin && ly.out_off[o] >= 0;
    const float* Wo = lin ? io.w + ly.wlin[o] : nullptr;
    const int ldw = ly.out_np[o] * n;
    if (lin) {   // At[c'][el*d3+m] = Vbar^L[e, c', o, m]
      for (int idx = tid; idx < TE * n * d3; idx += TP_T) {
        const int m = idx % d3, t2 = idx / d3, cp = t2 % n, el = t2 / n;
        At[cp * R + el * d3 + m] = (el < ne) ? io.vbar[((e0 + el) * n + cp) * ly.out_dim + ly.out_off[o] + m] : 0.f;
      }
    }
    for (int p = 0; p < ly.n_paths; ++p) {
      const int* pt = ly.path_tab + p * 8;
      if (pt[4] != o) continue;
      const int in_off = pt[0], d1 = pt[1], l2off = pt[2], pidx = pt[5], cb = pt[6], ce = pt[7];
      if (lin) {
        for (int idx = tid; idx < n * n; idx += TP_T) {   // Ws[c'][c] = W[c', pidx n + c]  (B2)
          const int cp = idx / n, c = idx - cp * n;
          Ws[idx] = Wo[(int64_t)cp * ldw + pidx * n + c];
        }
      }
      __syncthreads();
      // Tbar_p[c][r] = sum_c' At[c'][r] Ws[c'][c]   (+ sbar for the scalar paths, B4)
      const int ntr = R >> 2, ntc = n >> 2;
      for (int mt = tid; mt < ntr * ntc; mt += TP_T) {
        const int tr = mt % ntr, tc = mt / ntr;
        float a[4][4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) a[i][j] = 0.f;
        if (lin) {
          for (int k = 0; k < n; ++k) {
            const float4 av = *reinterpret_cast<const float4*>(At + k * R + tr * 4);
            const float4 bv = *reinterpret_cast<const float4*>(Ws + k * n + tc * 4);
            const float a4[4] = {av.x, av.y, av.z, av.w}, b4[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int j = 0; j < 4; ++j) a[i][j] = fmaf(a4[i], b4[j], a[i][j]);
          }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int r = tr * 4 + i, c = tc * 4 + j;
            float v = a[i][j];
            if (o == 0 && r < ne) v += io.sbar[(e0 + r) * (n * (ly.lmax + 1)) + pidx * n + c];   // d3 == 1: r == el
            Tt[c * R + r] = v;
          }
      }
      __syncthreads();
      // B5: Vbar^{L-1}[m1] += C Tbar[m3] Gamma[m2];  GE[m2] += C Tbar[m3] V[m1]
      for (int idx = tid; idx < TE * n; idx += TP_T) {
        const int el = idx % TE, c = idx / TE;
        if (el >= ne) continue;
        const int64_t e = e0 + el;
        const float* G = io.gamma + ((int64_t)io.e_center[e] * n + c) * ly.dsh + l2off;
        const float* Ye = Ys + el * 16;
        const float* tb = Tt + c * R + el * d3;
        float* vb = VB + (el * n + c) * ly.in_dim + in_off;
        float* gb = GE + (el * n + c) * ly.dsh + l2off;
        for (int q = cb; q < ce; ++q) {
          const int pk = ly.cg_idx[q];
          const int m1 = pk & 255, m2 = (pk >> 8) & 255, m3 = pk >> 16;
          const float ct = ly.cg_val[q] * tb[m3];
          vb[m1] = fmaf(ct, G[m2], vb[m1]);
          gb[m2] = fmaf(ct, tp_load_v(ly, io, e, c, in_off, d1, m1, Ye), gb[m2]);
        }
      }
      __syncthreads();
    }
  }
  for (int idx = tid; idx < ne * n * ly.in_dim; idx += TP_T) io.vbar_prev[e0 * n * ly.in_dim + idx] = VB[idx];
  for (int idx = tid; idx < ne * n * ly.dsh; idx += TP_T) io.ge[e0 * n * ly.dsh + idx] = GE[idx];
}

}  // namespace allegro
