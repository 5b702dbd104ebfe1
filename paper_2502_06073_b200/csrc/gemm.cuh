// gemm.cuh — contract of the edge-by-width GEMMs behind every dense linear map of the network (two-body MLP, W_init/W_env,
// latent MLPs, channel mixing, and their transposes in the analytic backward), PAPER.md:93 / Table 1:
//   C[e, n] = epi( sum_k pro(A[e, k]) * B(k, n) ),  A = [A0 | A1] (concat along k), B from the weight blob,
// with the fused prologues / epilogues below.  Kernels: gemm_tc.cu (chained MLPs and single linears, 3xTF32) and gemm_f16s.cu
// (wide linears, split fp16), all on tcgen05.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "device_math.cuh"
#include "model.h"

namespace allegro {

enum { PRO_NONE = 0, PRO_SILU = 1, PRO_SCALE_U = 2 };
enum { EPI_STORE = 0, EPI_GATHER2 = 1, EPI_Y_X = 2, EPI_RESIDUAL = 3, EPI_DSILU = 4, EPI_ACCUM = 5, EPI_SPLIT_RES = 6 };

struct GemmArgs {
  const int64_t* Mptr = nullptr;   // device: number of rows (active edges of the chunk)
  const float* A0 = nullptr; int lda0 = 0, K0 = 0;
  const float* A1 = nullptr; int lda1 = 0, K1 = 0;
  const float* W = nullptr; int ldw = 0, wtrans = 0;   // B(k,n) = wtrans ? W[k*ldw+n] : W[n*ldw+k]
  int N = 0;
  float* C = nullptr; int ldc = 0;
  float* C2 = nullptr; int ldc2 = 0;
  const float* aux = nullptr; int ldaux = 0;
  const float* geo = nullptr;       // [E][GEO_W]
  int pro = PRO_NONE, epi = EPI_STORE;
  float c_old = 0.f, c_new = 1.f;   // PRO_SCALE_U multiplies by c_new * u;  EPI_RESIDUAL / EPI_SPLIT_RES use both
  const float* Wg = nullptr; int ldwg = 0, S = 0;      // EPI_GATHER2: += Wg[n*ldwg + zi] + Wg[n*ldwg + S + zj]
  int split = 0;                     // EPI_SPLIT_RES: columns < split -> C (residual), >= split -> C2
  // optional row dot product fused into the chained epilogue (gemm_tc.cu; ignored by the single-GEMM kernels):
  //   dot_out[e] = (dot_accum ? dot_out[e] : 0) + dot_scale * sum_n pass[e, n] * (dotv ? dotv[n] : dotB[e, n])
  // where pass is the value the epilogue hands on (x^L for RESIDUAL, the accumulated sum for ACCUM, ...)
  // rows of the GEMM may be (edge, m) pairs of one irrep of an equivariant tensor stored as [e][comp][c] (tp_big.cuh):
  // M = *Mptr * m_mul rows; A0 row r / C row r live at tensor row (r / d3) * od + off + r % d3 when the map's d3 > 0
  int m_mul = 1;
  int amap_d3 = 0, amap_od = 0, amap_off = 0;
  int cmap_d3 = 0, cmap_od = 0, cmap_off = 0;     // EPI_STORE only
  float* dot_out = nullptr; const float* dotv = nullptr; const float* dotB = nullptr; int lddot = 0;
  float dot_scale = 1.f; int dot_accum = 0;
};

// one output element through the fused epilogue
__device__ __forceinline__ void gemm_epi(const GemmArgs& a, int64_t row, int n, float v, float u, int zi, int zj) {
  switch (a.epi) {
    case EPI_STORE: {
      const int64_t r2 = a.cmap_d3 ? (row / a.cmap_d3) * a.cmap_od + a.cmap_off + row % a.cmap_d3 : row;
      a.C[r2 * a.ldc + n] = v;
    } break;
    case EPI_GATHER2:
      a.C[row * a.ldc + n] = v + a.Wg[(int64_t)n * a.ldwg + zi] + a.Wg[(int64_t)n * a.ldwg + a.S + zj];
      break;
    case EPI_Y_X:
      a.C[row * a.ldc + n] = v; a.C2[row * a.ldc2 + n] = u * v; break;
    case EPI_RESIDUAL:
      a.C[row * a.ldc + n] = v;
      a.C2[row * a.ldc2 + n] = a.c_old * a.aux[row * a.ldaux + n] + a.c_new * u * v;
      break;
    case EPI_DSILU: a.C[row * a.ldc + n] = v * dsilu_f(a.aux[row * a.ldaux + n]); break;
    case EPI_ACCUM: a.C[row * a.ldc + n] += v; break;
    case EPI_SPLIT_RES:
      if (n < a.split) a.C[row * a.ldc + n] = a.c_old * a.aux[row * a.ldaux + n] + v;
      else a.C2[row * a.ldc2 + (n - a.split)] = v;
      break;
  }
}

// four consecutive output columns n..n+3 (n % 4 == 0, all < N, every leading dimension a multiple of 4).
// Returns the value a following chained stage consumes (gemm_chain.cu): the stored pre-activation for STORE / GATHER2,
// x = u v for Y_X, the new latent for RESIDUAL, v silu'(z) for DSILU, the accumulated sum for ACCUM.
__device__ __forceinline__ float4 gemm_epi4(const GemmArgs& a, int64_t row, int n, float4 v, float u, int zi, int zj) {
  auto ld4 = [](const float* p) { return *reinterpret_cast<const float4*>(p); };
  auto st4 = [](float* p, float4 x) { *reinterpret_cast<float4*>(p) = x; };
  switch (a.epi) {
    case EPI_STORE: {
      const int64_t r2 = a.cmap_d3 ? (row / a.cmap_d3) * a.cmap_od + a.cmap_off + row % a.cmap_d3 : row;
      st4(a.C + r2 * a.ldc + n, v);
      return v;
    }
    case EPI_GATHER2: {
      const float* g = a.Wg + (int64_t)n * a.ldwg;
      v.x += g[zi] + g[a.S + zj]; g += a.ldwg;
      v.y += g[zi] + g[a.S + zj]; g += a.ldwg;
      v.z += g[zi] + g[a.S + zj]; g += a.ldwg;
      v.w += g[zi] + g[a.S + zj];
      st4(a.C + row * a.ldc + n, v);
      return v;
    }
    case EPI_Y_X: {
      st4(a.C + row * a.ldc + n, v);
      const float4 x = make_float4(u * v.x, u * v.y, u * v.z, u * v.w);
      st4(a.C2 + row * a.ldc2 + n, x);
      return x;
    }
    case EPI_RESIDUAL: {
      st4(a.C + row * a.ldc + n, v);
      const float4 x = ld4(a.aux + row * a.ldaux + n);
      const float cu = a.c_new * u;
      const float4 r = make_float4(a.c_old * x.x + cu * v.x, a.c_old * x.y + cu * v.y, a.c_old * x.z + cu * v.z,
                                   a.c_old * x.w + cu * v.w);
      st4(a.C2 + row * a.ldc2 + n, r);
      return r;
    }
    case EPI_DSILU: {
      const float4 z = ld4(a.aux + row * a.ldaux + n);
      const float4 r = make_float4(v.x * dsilu_f(z.x), v.y * dsilu_f(z.y), v.z * dsilu_f(z.z), v.w * dsilu_f(z.w));
      st4(a.C + row * a.ldc + n, r);
      return r;
    }
    case EPI_ACCUM: {
      const float4 c = ld4(a.C + row * a.ldc + n);
      const float4 r = make_float4(c.x + v.x, c.y + v.y, c.z + v.z, c.w + v.w);
      st4(a.C + row * a.ldc + n, r);
      return r;
    }
    case EPI_SPLIT_RES:
      if (n < a.split) {
        const float4 x = ld4(a.aux + row * a.ldaux + n);
        st4(a.C + row * a.ldc + n, make_float4(a.c_old * x.x + v.x, a.c_old * x.y + v.y, a.c_old * x.z + v.z, a.c_old * x.w + v.w));
      } else {
        st4(a.C2 + row * a.ldc2 + (n - a.split), v);
      }
      return v;
  }
  return v;
}

void launch_gemm_tc(Model* m, const GemmArgs& a, int64_t m_cap, cudaStream_t st);   // gemm_tc.cu
// packed hi/lo B operand of a call site, built once and cached in the handle (gemm_tc.cu)
float* packed_weights(Model* m, const GemmArgs& a, cudaStream_t st, int* Npad, int* Kpad);
// a chain of up to 4 dependent GEMMs on the same 128-row tiles, activations kept in shared memory (gemm_chain.cu);
// returns false when the shapes do not fit (caller launches the stages one by one)
bool launch_gemm_chain(Model* m, const GemmArgs* stages, int n_stages, int64_t m_cap, cudaStream_t st);

// split-fp16 tcgen05 kernel for the wide linears (gemm_f16s.cu); false = shape / alignment outside what it takes
bool launch_gemm_f16s(Model* m, const GemmArgs& a, int64_t m_cap, cudaStream_t st);
const uint8_t* f16s_packed_weights(Model* m, const GemmArgs& a, cudaStream_t st, const float** out_scale);
// species columns of the first two-body matrix, transposed once and cached: WgT[z][n] = Wg[n * ldwg + z], z < 2S (gemm_tc.cu)
const float* transposed_species_columns(Model* m, const GemmArgs& a, cudaStream_t st);

inline void launch_gemm(Model* m, const GemmArgs& a, int64_t m_cap, cudaStream_t st) {
  if (m_cap <= 0) return;
  // wide linears: split-fp16 kernel; shapes or alignments it does not take (odd widths of small test networks): the per-linear
  // 3xTF32 kernel.  Both are tcgen05 kernels; there is no CUDA-core or CPU fallback.
  if (!launch_gemm_f16s(m, a, m_cap, st)) launch_gemm_tc(m, a, m_cap, st);
}

}  // namespace allegro
