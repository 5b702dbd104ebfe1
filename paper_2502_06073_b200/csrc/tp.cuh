// tp.cuh — F8/F9/F11 and B2/B5: the channel-wise Clebsch-Gordan tensor product V (x) Gamma of one layer, fused
// with the channel-mixing linear W_lin (forward) / its transpose (backward), so that the per-path product T is
// only ever held as a shared-memory tile ("64 tensor features with l=2 in full O(3) symmetry";
// readings A8, A9, A12).  The sparse coupling tensors are straight-line FMA code generated at build time
// (gen_tp.cpp -> tp_gen.cuh), one kernel instantiation per layer signature: V, Gamma and T stay in registers.
//
// Layouts (channel fastest, so that a warp's loads/stores are contiguous):
//   V[e][comp][c], Vbar[e][comp][c], GE[e][lm][c], Gamma[a][lm][c], winit/wenv/wbar[e][l*n + c], s[e][pidx*n + c].
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "device_math.cuh"
#include "model.h"
#include "tp_gen.cuh"

namespace allegro {

constexpr int TP_MAX_OUT = 8;
constexpr int TP_T = 256;

struct TpLayerDev {
  int n, lmax, dsh, in_dim, out_dim, n_paths, n_out, layer1, has_lin;
  const int* path_tab;     // [n_paths][8]: in_off, d1, l2off, d2, iro, pidx, -, -
  int out_d3[TP_MAX_OUT], out_off[TP_MAX_OUT], out_np[TP_MAX_OUT];
  long long wlin[TP_MAX_OUT];   // blob offsets of W_lin^{(l,p)}  [n, np*n]
};

struct TpIo {
  const int64_t* Mptr;
  const int* e_center;
  const float* geo;
  const float* gamma;      // [atoms, dsh, n]
  const float* vprev;      // [E, in_dim, n]      (layers >= 2)
  const float* winit; int ldwi;   // [E, .] first n_sc columns = W_init x0, column l*n + c   (layer 1)
  const float* w;          // weight blob
  float* s;                // [E, n_sc]   scalars (forward)
  float* vout;             // [E, out_dim, n]     (forward, has_lin)
  // backward
  const float* sbar;       // [E, n_sc]
  const float* vbar;       // [E, out_dim, n]  adjoint of V^L (has_lin)
  float* vbar_prev;        // [E, in_dim, n]
  float* ge;               // [E, dsh, n]  per-edge contribution to Gammabar
  float* wbar_init; int ldwb;   // layer 1: adjoint of (W_init x0)  [E, ., l*n + c]
  float* ybar;             // layer 1: [E, dsh]  adjoint of Y (accumulated)
};

__host__ __device__ __forceinline__ int tp_ldr(int R) { return (R % 8 == 0) ? R + 4 : R; }
__device__ __forceinline__ int l_of_lm(int k) { return (k >= 9) ? 3 : (k >= 4) ? 2 : (k >= 1) ? 1 : 0; }

// accessor of V^{L-1}[e, c, k]: layer 1 forms V^0 = (W_init x0)_{c,l} Y_lm on the fly (F5)
struct VAcc {
  const float* base; int stride; const float* Y; bool layer1;
  __device__ __forceinline__ float operator()(int k) const {
    if (layer1) return base[l_of_lm(k) * stride] * Y[k];
    return base[k * stride];
  }
};
struct GAcc {
  const float* base; int stride;
  __device__ __forceinline__ float operator()(int k) const { return base[k * stride]; }
};

// idx -> (idx / n, idx % n) without an integer division when n is a power of two (the usual case)
struct DivN {
  int n, sh, mask;
  __device__ __forceinline__ explicit DivN(int n_) : n(n_), sh(0), mask(((n_ & (n_ - 1)) == 0) ? n_ - 1 : -1) {
    while ((1 << sh) < n_) ++sh;
  }
  __device__ __forceinline__ void operator()(int idx, int* q, int* r) const {
    if (mask >= 0) { *q = idx >> sh; *r = idx & mask; }
    else { *q = idx / n; *r = idx - *q * n; }
  }
};
// small-range division by d3 in {1,3,5,7}: exact for idx < 2^14
struct DivS {
  int d, mul;
  __device__ __forceinline__ explicit DivS(int d_) : d(d_), mul((65536 + d_ - 1) / d_) {}
  __device__ __forceinline__ void operator()(int idx, int* q, int* r) const { *q = (idx * mul) >> 16; *r = idx - *q * d; }
};

// launchers (tp_kernels.cu)
void launch_tp_fwd(int sig, dim3 grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, int TE, int PC);
void launch_tp_bwd(int sig, dim3 grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, int TE, int d3max, int PC);
size_t tp3_smem_bytes(const TpLayerDev& tp, bool backward);
bool tp3_supported(const TpLayerDev& tp);
void launch_tp3(int sig, bool backward, int grid, cudaStream_t st, const TpLayerDev& tp, const TpIo& io);
struct TpBig;
bool tpbig_supported(const TpLayerDev& tp);
size_t tpbig_floats_per_edge(const TpLayerDev& tp);
bool launch_tpmix_fwd(Model* m, int sig, cudaStream_t st, const TpLayerDev& tp, const TpIo& io);   // tp_mix.cu
void launch_tpo(int sig, bool backward, int64_t m_cap, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, const TpBig& big);

constexpr int TP_MAXMT = 2;   // 4x4 micro-tiles per thread (forward): TE * d3 * n <= 8192
constexpr int TP_MAXP = 16;   // paths into one output irrep

// paths into output irrep o, in plan order (shared by the block)
__device__ __forceinline__ int tp_list_paths(const TpLayerDev& ly, int o, int* plist) {
  int np = 0;
  for (int p = 0; p < ly.n_paths; ++p)
    if (ly.path_tab[p * 8 + 4] == o && np < TP_MAXP) plist[np++] = p;
  return np;
}

// ---------------------------------------------------------------------------------------------------------
// forward: grid = (edge tiles, out irreps).  smem: Tt[PC n][ldR] | Ws[PC n][n] | Ys[TE][16]
// The paths into the irrep are processed PC at a time: T for the chunk is produced by the generated code, then one
// [R x PC n] x [PC n x n] product accumulates the channel mixing (F11).
// ---------------------------------------------------------------------------------------------------------
template <int SIG>
__global__ void __launch_bounds__(TP_T) k_tp_fwd(TpLayerDev ly, TpIo io, int TE, int PC) {
  extern __shared__ __align__(16) float sm[];
  __shared__ int plist[TP_MAXP], pidx_s[TP_MAXP];
  __shared__ int np_s;
  const int64_t M = *io.Mptr;
  const int64_t e0 = (int64_t)blockIdx.x * TE;
  if (e0 >= M) return;
  const int o = blockIdx.y;
  const DivN divn(ly.n);
  const int n = ly.n, d3 = ly.out_d3[o];
  const int R = TE * d3, ldR = tp_ldr(R);    // TE is a multiple of 4
  float* Tt = sm;                              // [PC n][ldR]
  float* Ws = Tt + PC * n * ldR;               // [PC n][n]  Ws[pi n + c][c'] = W[c', pidx n + c]
  float* Ys = Ws + PC * n * n;                 // [TE][16]
  const int tid = threadIdx.x;
  const int ne = (int)min((int64_t)TE, M - e0);
  const int nsc = n * (ly.lmax + 1);
  for (int t = tid; t < TE; t += TP_T) {
    float* y = Ys + t * 16;
    if (t < ne) { const float* gq = io.geo + (e0 + t) * GEO_W; sph_harm_rt(ly.lmax, gq[0], gq[1], gq[2], y); }
  }
  if (tid == 0) {
    np_s = tp_list_paths(ly, o, plist);
    for (int k = 0; k < np_s; ++k) pidx_s[k] = ly.path_tab[plist[k] * 8 + 5];
  }
  const bool lin = ly.has_lin && ly.out_off[o] >= 0;
  const int ntr = R >> 2, ntc = n >> 2, nmt = ntr * ntc;
  const DivS divd3(d3);
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
  const int np = np_s;
  for (int ch = 0; ch < np; ch += PC) {
    const int cnt = min(PC, np - ch);
    // T_p[e, c, m3] for the tile and the paths of the chunk: one (edge, channel) pair per thread and iteration, all
    // paths of the chunk for that pair back to back (V, Gamma addresses formed once)
    for (int idx = tid; idx < TE * n; idx += TP_T) {
      int el, c;
      divn(idx, &el, &c);
      float* dst0 = Tt + c * ldR + el * d3;
      if (el >= ne) {
        for (int pi = 0; pi < cnt; ++pi)
          for (int m = 0; m < d3; ++m) dst0[pi * n * ldR + m] = 0.f;
        continue;
      }
      const int64_t e = e0 + el;
      VAcc V{ly.layer1 ? io.winit + e * io.ldwi + c : io.vprev + e * ly.in_dim * n + c, n, Ys + el * 16, ly.layer1 != 0};
      GAcc G{io.gamma + (int64_t)io.e_center[e] * ly.dsh * n + c, n};
      for (int pi = 0; pi < cnt; ++pi) {
        const int p = plist[ch + pi];
        float* dst = dst0 + pi * n * ldR;
        float t0 = 0.f;
        tpgen::tp_path_fwd<SIG>(p, V, G, [&](int m, float v) { dst[m] = v; if (m == 0) t0 = v; });
        if (o == 0) io.s[e * nsc + pidx_s[ch + pi] * n + c] = t0;   // F9: path-major, then channel
      }
    }
    if (lin) {
      for (int idx = tid; idx < cnt * n * n; idx += TP_T) {
        int t2, c, pi, cp;
        divn(idx, &t2, &c);
        divn(t2, &pi, &cp);                                              // coalesced along c
        Ws[(pi * n + c) * n + cp] = Wo[(int64_t)cp * ldw + pidx_s[ch + pi] * n + c];
      }
    }
    __syncthreads();
    if (lin) {
      const int K = cnt * n;
#pragma unroll
      for (int q = 0; q < TP_MAXMT; ++q) {
        const int mt = tid + q * TP_T;
        if (mt < nmt) {
          const int tr = mt % ntr, tc = mt / ntr;
#pragma unroll 4
          for (int k = 0; k < K; ++k) {
            const float4 av = *reinterpret_cast<const float4*>(Tt + k * ldR + tr * 4);
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
          int el, m;
          divd3(tr * 4 + i, &el, &m);
          if (el < ne)
            *reinterpret_cast<float4*>(io.vout + ((e0 + el) * ly.out_dim + ooff + m) * n + tc * 4) =
                make_float4(acc[q][i][0], acc[q][i][1], acc[q][i][2], acc[q][i][3]);
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// backward: one block per TE edges, all out irreps and paths.
// smem: VB[TE][in_dim][n] | GE[TE][dsh][n] | At[n][ldRmax] | Tt[PC n][ldRmax] | Ws[n][PC n] | Ys[TE][16]
// Layer 1 also applies B8 in place (adjoint of V^0 = (W_init x0) Y): wbar_init and the Ybar contribution are formed
// from the shared-memory Vbar^0 tile, which is then never written to global memory.
// ---------------------------------------------------------------------------------------------------------
template <int SIG>
__global__ void __launch_bounds__(TP_T) k_tp_bwd(TpLayerDev ly, TpIo io, int TE, int d3max, int PC) {
  extern __shared__ __align__(16) float sm[];
  __shared__ int plist[TP_MAXP], pidx_s[TP_MAXP];
  __shared__ int np_s;
  const int64_t M = *io.Mptr;
  const int64_t e0 = (int64_t)blockIdx.x * TE;
  if (e0 >= M) return;
  const DivN divn(ly.n);
  const int n = ly.n, ldRmax = tp_ldr(TE * d3max) + 4;
  float* VB = sm;
  float* GE = VB + TE * n * ly.in_dim;
  float* At = GE + TE * n * ly.dsh;
  float* Tt = At + n * ldRmax;
  float* Ws = Tt + PC * n * ldRmax;
  float* Ys = Ws + PC * n * n;
  const int tid = threadIdx.x;
  const int ne = (int)min((int64_t)TE, M - e0);
  const int nsc = n * (ly.lmax + 1);
  for (int t = tid; t < TE; t += TP_T)
    if (t < ne) { const float* gq = io.geo + (e0 + t) * GEO_W; sph_harm_rt(ly.lmax, gq[0], gq[1], gq[2], Ys + t * 16); }
  for (int idx = tid; idx < TE * n * (ly.in_dim + ly.dsh); idx += TP_T) VB[idx] = 0.f;   // VB and GE are adjacent
  for (int o = 0; o < ly.n_out; ++o) {
    const int d3 = ly.out_d3[o], R = TE * d3, ldR = tp_ldr(R);
    const bool lin = ly.has_lin && ly.out_off[o] >= 0;
    if (!lin && o != 0) continue;
    const float* Wo = lin ? io.w + ly.wlin[o] : nullptr;
    const int ldw = ly.out_np[o] * n;
    __syncthreads();
    if (tid == 0) {
      np_s = tp_list_paths(ly, o, plist);
      for (int k = 0; k < np_s; ++k) pidx_s[k] = ly.path_tab[plist[k] * 8 + 5];
    }
    if (lin) {   // At[c'][el*d3+m] = Vbar^L[e, o, m, c']
      const DivS divd3(d3);
      for (int idx = tid; idx < TE * n * d3; idx += TP_T) {
        int row, cp, el, m;
        divn(idx, &row, &cp);
        divd3(row, &el, &m);
        At[cp * ldR + row] = (el < ne) ? io.vbar[((e0 + el) * ly.out_dim + ly.out_off[o] + m) * n + cp] : 0.f;
      }
    }
    __syncthreads();
    const int np = np_s;
    for (int ch = 0; ch < np; ch += PC) {
      const int cnt = min(PC, np - ch), NC = cnt * n;
      if (lin) {
        for (int idx = tid; idx < n * NC; idx += TP_T) {   // Ws[c'][pi n + c] = W[c', pidx n + c]  (B2)
          int t2, c;
          divn(idx, &t2, &c);
          const int cp = t2 / cnt, pi = t2 - cp * cnt;
          Ws[cp * NC + pi * n + c] = Wo[(int64_t)cp * ldw + pidx_s[ch + pi] * n + c];
        }
      }
      __syncthreads();
      // Tbar_p[c][r] = sum_c' At[c'][r] Ws[c'][pi n + c]   (+ sbar for the scalar paths, B4)
      const int ntr = R >> 2, ntc = NC >> 2;
      for (int mt = tid; mt < ntr * ntc; mt += TP_T) {
        const int tr = mt % ntr, tc = mt / ntr;
        float a[4][4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) a[i][j] = 0.f;
        if (lin) {
#pragma unroll 4
          for (int k = 0; k < n; ++k) {
            const float4 av = *reinterpret_cast<const float4*>(At + k * ldR + tr * 4);
            const float4 bv = *reinterpret_cast<const float4*>(Ws + k * NC + tc * 4);
            const float a4[4] = {av.x, av.y, av.z, av.w}, b4[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int j = 0; j < 4; ++j) a[i][j] = fmaf(a4[i], b4[j], a[i][j]);
          }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int col = tc * 4 + j;             // pi n + c
          float4 v = make_float4(a[0][j], a[1][j], a[2][j], a[3][j]);
          if (o == 0) {   // d3 == 1: row r == el
            int pi, c;
            divn(col, &pi, &c);
            const int64_t so = (int64_t)pidx_s[ch + pi] * n + c;
            const int r = tr * 4;
            if (r < ne) v.x += io.sbar[(e0 + r) * nsc + so];
            if (r + 1 < ne) v.y += io.sbar[(e0 + r + 1) * nsc + so];
            if (r + 2 < ne) v.z += io.sbar[(e0 + r + 2) * nsc + so];
            if (r + 3 < ne) v.w += io.sbar[(e0 + r + 3) * nsc + so];
          }
          *reinterpret_cast<float4*>(Tt + col * ldR + tr * 4) = v;
        }
      }
      __syncthreads();
      // B5: Vbar^{L-1}[m1] += C Tbar[m3] Gamma[m2];  GE[m2] += C Tbar[m3] V[m1].  Paths of a chunk are applied one after
      // the other by the same thread (pair (el, c) fixed), so the shared-memory accumulation has no race.
      for (int idx = tid; idx < TE * n; idx += TP_T) {
        int el, c;
        divn(idx, &el, &c);
        if (el >= ne) continue;
        const int64_t e = e0 + el;
        VAcc V{ly.layer1 ? io.winit + e * io.ldwi + c : io.vprev + e * ly.in_dim * n + c, n, Ys + el * 16, ly.layer1 != 0};
        GAcc G{io.gamma + (int64_t)io.e_center[e] * ly.dsh * n + c, n};
        float* vb = VB + el * ly.in_dim * n + c;
        float* gb = GE + el * ly.dsh * n + c;
        for (int pi = 0; pi < cnt; ++pi) {
          const float* tb = Tt + (pi * n + c) * ldR + el * d3;
          tpgen::tp_path_bwd<SIG>(plist[ch + pi], V, G, [&](int m) { return tb[m]; }, [&](int k, float v) { vb[k * n] += v; },
                                  [&](int k, float v) { gb[k * n] += v; });
        }
      }
    }
  }
  __syncthreads();
  for (int idx = tid; idx < ne * n * ly.dsh; idx += TP_T) io.ge[e0 * n * ly.dsh + idx] = GE[idx];
  if (!ly.layer1) {
    for (int idx = tid; idx < ne * n * ly.in_dim; idx += TP_T) io.vbar_prev[e0 * n * ly.in_dim + idx] = VB[idx];
  } else {
    // B8 (in_dim == dsh): wbar_init[e, l, c] = sum_m Vbar0[e, lm, c] Y_lm(e)
    const int nl1 = ly.lmax + 1;
    for (int idx = tid; idx < ne * nsc; idx += TP_T) {
      int t2, c;
      divn(idx, &t2, &c);
      const int el = t2 / nl1, l = t2 - el * nl1;
      const float* vb = VB + (el * ly.dsh + l * l) * n + c;
      const float* Y = Ys + el * 16 + l * l;
      float sacc = 0.f;
      for (int mm = 0; mm < 2 * l + 1; ++mm) sacc = fmaf(vb[mm * n], Y[mm], sacc);
      io.wbar_init[(e0 + el) * io.ldwb + l * n + c] = sacc;
    }
    // Ybar[e, lm] += sum_c (W_init x0)[e, l, c] Vbar0[e, lm, c]   (channel index rotated per thread: no bank conflicts)
    for (int idx = tid; idx < ne * ly.dsh; idx += TP_T) {
      const int lm = idx % ly.dsh, el = idx / ly.dsh;
      const float* vb = VB + (el * ly.dsh + lm) * n;
      const float* wi = io.winit + (e0 + el) * io.ldwi + l_of_lm(lm) * n;
      float sacc = 0.f;
      int c = tid % n;
      for (int cc = 0; cc < n; ++cc) {
        sacc = fmaf(wi[c], vb[c], sacc);
        if (++c == n) c = 0;
      }
      io.ybar[(e0 + el) * ly.dsh + lm] += sacc;
    }
  }
}

}  // namespace allegro
