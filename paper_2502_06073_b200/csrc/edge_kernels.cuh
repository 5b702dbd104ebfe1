// edge_kernels.cuh — per-edge and per-row (centre atom) kernels of the forward and backward pass.
// Steps refer to SURVEY.md 8c (F1-F12, B1-B12); PAPER.md:93 / :9 are the paper passages behind them.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "device_math.cuh"
#include "model.h"

namespace allegro {

struct ListView {
  const int64_t* rowptr;   // [N+1] list rows
  const uint64_t* keys;    // [E_list] packed (j, s)
  const int* revpos;       // [E_list]
  double H[9];             // cell, rows = lattice vectors
};

__device__ __forceinline__ void decode_key(uint64_t key, int* j, int* sx, int* sy, int* sz) {
  *j = (int)(key >> 24);
  *sx = (int)((key >> 16) & 255) - 128; *sy = (int)((key >> 8) & 255) - 128; *sz = (int)(key & 255) - 128;
}

// Cartesian component c of the image shift s: (s_1 a_1c + s_2 a_2c) + s_3 a_3c, fp64, no FMA contraction (reading A27).  For a
// diagonal H the two added products are exact zeros: the value is s_c L_c bit for bit, the expression of A16.
__device__ __forceinline__ double image_shift(const double* H, int c, int sx, int sy, int sz) {
  return __dadd_rn(__dadd_rn(__dmul_rn((double)sx, H[c]), __dmul_rn((double)sy, H[3 + c])), __dmul_rn((double)sz, H[6 + c]));
}
__device__ __forceinline__ double edge_d2(const double* __restrict__ pos, int64_t i, uint64_t key, const double* H,
                                          double* dx, double* dy, double* dz, int* jout) {
  int j, sx, sy, sz;
  decode_key(key, &j, &sx, &sy, &sz);
  *jout = j;
  // A16: same expression order as the list criterion, fp64, no FMA contraction
  *dx = __dadd_rn(__dsub_rn(pos[3 * (int64_t)j], pos[3 * i]), image_shift(H, 0, sx, sy, sz));
  *dy = __dadd_rn(__dsub_rn(pos[3 * (int64_t)j + 1], pos[3 * i + 1]), image_shift(H, 1, sx, sy, sz));
  *dz = __dadd_rn(__dsub_rn(pos[3 * (int64_t)j + 2], pos[3 * i + 2]), image_shift(H, 2, sx, sy, sz));
  return __dadd_rn(__dadd_rn(__dmul_rn(*dx, *dx), __dmul_rn(*dy, *dy)), __dmul_rn(*dz, *dz));
}

// stale-list test (A22) + species range check: one thread per atom
__global__ void k_check_inputs(const double* __restrict__ pos, const double* __restrict__ r_build, const int* __restrict__ species,
                               int64_t N, double half_skin2, int n_species, int* flags) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const double dx = __dsub_rn(pos[3 * i], r_build[3 * i]), dy = __dsub_rn(pos[3 * i + 1], r_build[3 * i + 1]), dz = __dsub_rn(pos[3 * i + 2], r_build[3 * i + 2]);
  const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));   // as the oracle: no FMA contraction
  if (d2 > half_skin2 && !flags[FLAG_HALT]) flags[FLAG_STALE] = 1;   // halted integrator: the host rebuilds and redoes this evaluation
  int z = species[i];
  if (z < 0 || z >= n_species) flags[FLAG_SPECIES] = 1;
}

// a-2 (first half): active-edge compaction (A11: edges with r >= r_c contribute exactly zero and are dropped).
// One warp per centre atom of the chunk [a0, a1).  MODE 0 counts, MODE 1 fills the chunk-local edge arrays,
// computes the edge geometry in fp64 (rounded to fp32 once) and zeroes g_list for the inactive list edges.
template <int MODE>
__global__ void k_active(const double* __restrict__ pos, const int* __restrict__ species, ListView lv, int64_t a0, int64_t a1,
                         double rc, int poly_p, int n_bessel, int* __restrict__ act_cnt, const int64_t* __restrict__ rowptr_c,
                         int* __restrict__ e_center, int* __restrict__ e_j, int64_t* __restrict__ e_lidx,
                         float* __restrict__ geo, float* __restrict__ bes, float* __restrict__ g_list, int64_t cap_edges, int* flags) {
  const int lane = threadIdx.x & 31;
  const int64_t a = a0 + (((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  if (a >= a1) return;
  const int64_t b = lv.rowptr[a], e = lv.rowptr[a + 1];
  const double rc2 = rc * rc;
  int total = 0;
  const int64_t base = MODE ? rowptr_c[a - a0] : 0;
  const int zi = MODE ? species[a] : 0;
  for (int64_t k0 = b; k0 < e; k0 += 32) {
    const int64_t k = k0 + lane;
    bool act = false;
    double dx = 0, dy = 0, dz = 0, d2 = 0;
    int j = 0;
    if (k < e) {
      d2 = edge_d2(pos, a, lv.keys[k], lv.H, &dx, &dy, &dz, &j);
      act = d2 < rc2;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, act);
    if (MODE == 1 && k < e) {
      if (!act) {
        g_list[3 * k] = 0.f; g_list[3 * k + 1] = 0.f; g_list[3 * k + 2] = 0.f;
      } else {
        const int64_t dst = base + total + __popc(bal & ((1u << lane) - 1u));
        if (dst < cap_edges) {
          const double r = sqrt(d2), inv = 1.0 / r;
          const double x = r / rc;
          double u, dudx;
          envelope_d(x, poly_p, &u, &dudx);
          e_center[dst] = (int)(a - a0);
          e_j[dst] = j;
          e_lidx[dst] = k;
          float* gq = geo + dst * GEO_W;
          gq[0] = (float)(dx * inv); gq[1] = (float)(dy * inv); gq[2] = (float)(dz * inv);
          gq[3] = (float)r; gq[4] = (float)u; gq[5] = (float)(dudx / rc);
          gq[6] = __int_as_float(zi); gq[7] = __int_as_float(species[j]);
          // F2: b_n = (2/rc) sin(n pi r/rc)/r * u
          const double pref = 2.0 / rc * inv * u, w = 3.14159265358979323846 * x;
          for (int n = 1; n <= n_bessel; ++n) bes[dst * n_bessel + (n - 1)] = (float)(pref * sin(n * w));
        } else {
          flags[FLAG_ERR_CAP] = 2;   // unreachable after k_ws_check / k_ws_clamp; kept as a guard
        }
      }
    }
    total += __popc(bal);
  }
  if (MODE == 0 && lane == 0) act_cnt[a - a0] = total;
}

// Activation-workspace guard: when the chunk holds more active edges than the workspace, the chunk is emptied (every row
// offset 0: all edge kernels see M = 0 and do nothing), the error is flagged and the integrator halted; the host re-sizes.
__global__ void k_ws_check(const int64_t* rowptr_c, int64_t na, int64_t cap_edges, int* flags) {
  if (rowptr_c[na] > cap_edges) { flags[FLAG_ERR_CAP] = 2; flags[FLAG_HALT] = 1; }
}
__global__ void k_ws_clamp(int64_t* rowptr_c, int64_t na, const int* flags) {
  if (flags[FLAG_ERR_CAP] != 2) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= na) rowptr_c[i] = 0;
}

// F7: Gamma_i[lm, c] = Nbar^-1/2 sum_{e in row(i)} w[e, l, c] Y_lm(rhat_e).  One block per centre atom.  A thread owns a
// channel c and every (256 / n)-th edge of the row: it forms w[e, l, c] Y_lm(e) for all lm in registers and sums over its
// edges; the 256 / n partial sums per output are then added in a fixed order through shared memory (deterministic, no
// atomics).  w[e][l*n + c] and Gamma[a][lm][c] are read / written contiguously in c.
constexpr int GAMMA_T = 256;
template <int LMAX>
__global__ void __launch_bounds__(GAMMA_T) k_gamma_t(const int64_t* __restrict__ rowptr_c, const float* __restrict__ geo,
                                                    const float* __restrict__ w, int ldw, int n, float inv_sqrt_navg,
                                                    float* __restrict__ gamma, int64_t n_atoms) {
  constexpr int DSH = (LMAX + 1) * (LMAX + 1);
  __shared__ float red[GAMMA_T * (DSH + 1)];
  const int64_t a = blockIdx.x;
  if (a >= n_atoms) return;
  const int64_t b = rowptr_c[a], e = rowptr_c[a + 1];
  const int epb = GAMMA_T / n;                  // edges in flight per pass (n <= 256)
  const int c = threadIdx.x % n, grp = threadIdx.x / n;
  float acc[DSH];
#pragma unroll
  for (int k = 0; k < DSH; ++k) acc[k] = 0.f;
  if (grp < epb) {
    for (int64_t k = b + grp; k < e; k += epb) {
      const float* gq = geo + k * GEO_W;
      float Y[16];
      sph_harm<LMAX>(gq[0], gq[1], gq[2], Y);
      const float* wk = w + k * ldw + c;
#pragma unroll
      for (int l = 0; l <= LMAX; ++l) {
        const float wl = wk[l * n];
#pragma unroll
        for (int mm = 0; mm < 2 * l + 1; ++mm) acc[l * l + mm] = fmaf(wl, Y[l * l + mm], acc[l * l + mm]);
      }
    }
  }
#pragma unroll
  for (int k = 0; k < DSH; ++k) red[threadIdx.x * (DSH + 1) + k] = acc[k];
  __syncthreads();
  const int nout = n * DSH;
  for (int o = threadIdx.x; o < nout; o += GAMMA_T) {
    const int lm = o / n, cc = o - lm * n;
    float s = 0.f;
    for (int g2 = 0; g2 < epb; ++g2) s += red[(g2 * n + cc) * (DSH + 1) + lm];
    gamma[a * nout + o] = inv_sqrt_navg * s;
  }
}
inline void launch_gamma(const int64_t* rowptr_c, const float* geo, const float* w, int ldw, int n, int lmax, float inv_sqrt_navg,
                         float* gamma, int64_t n_atoms, cudaStream_t st) {
  const unsigned g = (unsigned)n_atoms;
  switch (lmax) {
    case 0: k_gamma_t<0><<<g, GAMMA_T, 0, st>>>(rowptr_c, geo, w, ldw, n, inv_sqrt_navg, gamma, n_atoms); break;
    case 1: k_gamma_t<1><<<g, GAMMA_T, 0, st>>>(rowptr_c, geo, w, ldw, n, inv_sqrt_navg, gamma, n_atoms); break;
    case 2: k_gamma_t<2><<<g, GAMMA_T, 0, st>>>(rowptr_c, geo, w, ldw, n, inv_sqrt_navg, gamma, n_atoms); break;
    default: k_gamma_t<3><<<g, GAMMA_T, 0, st>>>(rowptr_c, geo, w, ldw, n, inv_sqrt_navg, gamma, n_atoms); break;
  }
}

// B5 (row reduction) + B6: Gammabar_i = sum_row GE[e], then for every edge of the row
//   wbar[e,l,c] = Nbar^-1/2 sum_m Gammabar[l,m,c] Y_lm(e);   Ybar[e,lm] += Nbar^-1/2 sum_c w[e,l,c] Gammabar[lm,c].
// One block per centre atom, Gammabar kept in shared memory ([lm][n+1], padded against bank conflicts).  lmax and (for
// n = 8, 16, 32) the channel count are compile-time constants: the kernel is issue-bound on address arithmetic otherwise.
template <int LMAX, int NCH>
__global__ void __launch_bounds__(128) k_gammabar_t(const int64_t* __restrict__ rowptr_c, const float* __restrict__ geo,
                                                   const float* __restrict__ ge, const float* __restrict__ w, int ldw, int n_rt,
                                                   float inv_sqrt_navg, float* __restrict__ wbar, int ldwb, float* __restrict__ ybar,
                                                   int64_t n_atoms) {
  extern __shared__ float sm[];
  constexpr int DSH = (LMAX + 1) * (LMAX + 1);
  const int n = NCH ? NCH : n_rt;
  const int64_t a = blockIdx.x;
  if (a >= n_atoms) return;
  const int nout = n * DSH, ldg = n + 1;
  float* Gb = sm;              // [DSH][n+1]
  const int64_t b = rowptr_c[a], e = rowptr_c[a + 1];
  const int len = (int)(e - b);
  if (len == 0) return;
  for (int o = threadIdx.x; o < nout; o += 128) {
    float s = 0.f;
    const float* gp = ge + b * nout + o;
    for (int k = 0; k < len; ++k) s += gp[(int64_t)k * nout];
    const int lm = o / n, c = o - lm * n;
    Gb[lm * ldg + c] = s * inv_sqrt_navg;
  }
  __syncthreads();
  // wbar: one (edge, channel) pair per thread and iteration
  for (int idx = threadIdx.x; idx < len * n; idx += 128) {
    const int kk = idx / n, c = idx - kk * n;
    const int64_t k = b + kk;
    const float* gq = geo + k * GEO_W;
    float Y[16];
    sph_harm<LMAX>(gq[0], gq[1], gq[2], Y);
    float* wo = wbar + k * ldwb + c;
#pragma unroll
    for (int l = 0; l <= LMAX; ++l) {
      float s = 0.f;
#pragma unroll
      for (int mm = 0; mm < 2 * l + 1; ++mm) s = fmaf(Gb[(l * l + mm) * ldg + c], Y[l * l + mm], s);
      wo[l * n] = s;
    }
  }
  // Ybar: one (edge, lm) pair per thread and iteration
  for (int idx = threadIdx.x; idx < len * DSH; idx += 128) {
    const int kk = idx / DSH, lm = idx - kk * DSH;
    const int64_t k = b + kk;
    const int l = (lm >= 9) ? 3 : (lm >= 4) ? 2 : (lm >= 1) ? 1 : 0;
    const float* wk = w + k * ldw + l * n;
    const float* g = Gb + lm * ldg;
    float s = 0.f;
    if (NCH) {
#pragma unroll
      for (int c = 0; c < (NCH ? NCH : 1); c += 4) {
        const float4 w4 = *reinterpret_cast<const float4*>(wk + c);
        s = fmaf(w4.x, g[c], fmaf(w4.y, g[c + 1], fmaf(w4.z, g[c + 2], fmaf(w4.w, g[c + 3], s))));
      }
    } else {
      for (int c = 0; c < n; ++c) s = fmaf(wk[c], g[c], s);
    }
    ybar[k * DSH + lm] += s;
  }
}

template <int LMAX>
static void launch_gammabar_l(unsigned grid, size_t smem, cudaStream_t st, const int64_t* rowptr_c, const float* geo, const float* ge,
                              const float* w, int ldw, int n, float inv, float* wbar, int ldwb, float* ybar, int64_t na) {
  const bool vec = (ldw % 4 == 0) && ((((uintptr_t)w) & 15) == 0);
  if (n == 8 && vec) k_gammabar_t<LMAX, 8><<<grid, 128, smem, st>>>(rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na);
  else if (n == 16 && vec) k_gammabar_t<LMAX, 16><<<grid, 128, smem, st>>>(rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na);
  else if (n == 32 && vec) k_gammabar_t<LMAX, 32><<<grid, 128, smem, st>>>(rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na);
  else k_gammabar_t<LMAX, 0><<<grid, 128, smem, st>>>(rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na);
}
inline void launch_gammabar(const int64_t* rowptr_c, const float* geo, const float* ge, const float* w, int ldw, int n, int lmax,
                            float inv, float* wbar, int ldwb, float* ybar, int64_t na, cudaStream_t st) {
  const int dsh = (lmax + 1) * (lmax + 1);
  const size_t smem = (size_t)(dsh * (n + 1) + 16) * sizeof(float);
  const unsigned grid = (unsigned)na;
  switch (lmax) {
    case 0: launch_gammabar_l<0>(grid, smem, st, rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na); break;
    case 1: launch_gammabar_l<1>(grid, smem, st, rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na); break;
    case 2: launch_gammabar_l<2>(grid, smem, st, rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na); break;
    default: launch_gammabar_l<3>(grid, smem, st, rowptr_c, geo, ge, w, ldw, n, inv, wbar, ldwb, ybar, na); break;
  }
}

// active-edge counter of a force call, summed over its atom chunks
__global__ void k_add_count(const int64_t* __restrict__ cnt, int64_t* __restrict__ total) { *total += *cnt; }

// B1 fused with the first B3 dot: xbar^{NL}[e, :] = sigma_{Z_i} w_eff and ubar[e] = c_new (xbar^{NL}_e . y^{NL}_e).  One warp per edge.
__global__ void k_xbar_init_dot(const int64_t* __restrict__ Mptr, const float* __restrict__ geo, const float* __restrict__ sigma,
                                const float* __restrict__ weff, int D, const float* __restrict__ y, float c_new,
                                float* __restrict__ xbar, float* __restrict__ ubar) {
  const int lane = threadIdx.x & 31;
  const int64_t e = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (e >= *Mptr) return;
  const float sg = sigma[__float_as_int(geo[e * GEO_W + 6])];
  float s = 0.f;
  for (int d = lane; d < D; d += 32) {
    const float xb = sg * weff[d];
    xbar[e * D + d] = xb;
    s = fmaf(xb, y[e * D + d], s);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if (lane == 0) ubar[e] = c_new * s;
}

// Same, D a multiple of 4 with D / 4 a power of two <= 32: D / 4 threads per edge, 128-bit accesses.
__global__ void k_xbar_init_dot4(const int64_t* __restrict__ Mptr, const float* __restrict__ geo, const float* __restrict__ sigma,
                                 const float* __restrict__ weff, int D, const float* __restrict__ y, float c_new,
                                 float* __restrict__ xbar, float* __restrict__ ubar) {
  const int q4 = D >> 2;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t e = idx / q4;
  const int q = (int)(idx - e * q4);
  const bool valid = e < *Mptr;
  float s = 0.f;
  if (valid) {
    const float sg = sigma[__float_as_int(geo[e * GEO_W + 6])];
    const float4 w4 = *reinterpret_cast<const float4*>(weff + 4 * q);
    const float4 y4 = *reinterpret_cast<const float4*>(y + e * D + 4 * q);
    const float4 xb = make_float4(sg * w4.x, sg * w4.y, sg * w4.z, sg * w4.w);
    *reinterpret_cast<float4*>(xbar + e * D + 4 * q) = xb;
    s = fmaf(xb.x, y4.x, fmaf(xb.y, y4.y, fmaf(xb.z, y4.z, xb.w * y4.w)));
  }
  for (int d = q4 >> 1; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if (q == 0 && valid) ubar[e] = c_new * s;
}

// F12 with eps_e already formed by the GEMM epilogue: E_i = sigma_{Z_i} sum_row eps_e + mu_{Z_i}.  One warp per centre atom.
__global__ void k_readout_eps(const int64_t* __restrict__ rowptr_c, const float* __restrict__ eps, const int* __restrict__ species,
                              int64_t a0, int64_t n_atoms, const float* __restrict__ sigma, const float* __restrict__ mu,
                              float* __restrict__ e_atom) {
  const int lane = threadIdx.x & 31;
  const int64_t a = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n_atoms) return;
  float s = 0.f;
  for (int64_t k = rowptr_c[a] + lane; k < rowptr_c[a + 1]; k += 32) s += eps[k];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if (lane == 0) {
    const int z = species[a0 + a];
    e_atom[a0 + a] = sigma[z] * s + mu[z];
  }
}

// out[e] (+)= scale * dot(A[e,:], B[e,:])   (ubar contributions of B3 and B9).  One warp per edge.
__global__ void k_rowdot(const int64_t* __restrict__ Mptr, const float* __restrict__ A, const float* __restrict__ B, int D,
                         float scale, int accumulate, float* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t e = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (e >= *Mptr) return;
  float s = 0.f;
  for (int d = lane; d < D; d += 32) s = fmaf(A[e * D + d], B[e * D + d], s);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if (lane == 0) out[e] = (accumulate ? out[e] : 0.f) + scale * s;
}

// F12: eps_e = w_eff . x^{NL}_e;  E_i = sigma_{Z_i} sum_row eps_e + mu_{Z_i}.  One warp per centre atom.
__global__ void k_readout(const int64_t* __restrict__ rowptr_c, const float* __restrict__ x, int D, const float* __restrict__ weff,
                          const int* __restrict__ species, int64_t a0, int64_t n_atoms, const float* __restrict__ sigma,
                          const float* __restrict__ mu, float* __restrict__ e_atom) {
  const int lane = threadIdx.x & 31;
  const int64_t a = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (a >= n_atoms) return;
  float s = 0.f;
  for (int64_t k = rowptr_c[a]; k < rowptr_c[a + 1]; ++k)
    for (int d = lane; d < D; d += 32) s = fmaf(x[k * D + d], weff[d], s);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if (lane == 0) {
    const int z = species[a0 + a];
    e_atom[a0 + a] = sigma[z] * s + mu[z];
  }
}

// B10 + B11: g_e = rbar rhat + (1/r)(I - rhat rhat^T) sum_lm Ybar_lm grad Y_lm, written at the edge's list position.
__global__ void k_edge_grad(const int64_t* __restrict__ Mptr, const float* __restrict__ geo, const float* __restrict__ bes,
                            const float* __restrict__ bbar, const float* __restrict__ ubar, const float* __restrict__ ybar,
                            const int64_t* __restrict__ e_lidx, int n_bessel, int lmax, float rc, float* __restrict__ g_list) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= *Mptr) return;
  const float* gq = geo + e * GEO_W;
  const float x = gq[0], y = gq[1], z = gq[2], r = gq[3], u = gq[4], du = gq[5];
  const int dsh = (lmax + 1) * (lmax + 1);
  // d b_n/dr = (2/rc)(k cos(kr)/r - sin(kr)/r^2) u + B_n du  with B_n u = b_n  =>  = (2/rc) k cos(kr) u / r - b_n / r + (b_n/u) du
  float rbar = ubar[e] * du;
  const float inv_r = 1.0f / r, pref = 2.0f / rc;
  for (int n = 1; n <= n_bessel; ++n) {
    const float k = n * 3.14159265358979f / rc;
    float sn, cs;
    sincosf(k * r, &sn, &cs);
    const float Bn = pref * sn * inv_r;
    const float dBn = pref * (k * cs * inv_r - sn * inv_r * inv_r);
    rbar = fmaf(bbar[e * n_bessel + (n - 1)], dBn * u + Bn * du, rbar);
  }
  float Yb[16], t[3];
  for (int q = 0; q < dsh; ++q) Yb[q] = ybar[e * dsh + q];
  sph_harm_vjp(lmax, x, y, z, Yb, t);
  const float tr = t[0] * x + t[1] * y + t[2] * z;
  const int64_t k = e_lidx[e];
  g_list[3 * k] = rbar * x + (t[0] - tr * x) * inv_r;
  g_list[3 * k + 1] = rbar * y + (t[1] - tr * y) * inv_r;
  g_list[3 * k + 2] = rbar * z + (t[2] - tr * z) * inv_r;
}

// B12: F_i = sum_{e in row(i)} (g_e - g_rev(e)), accumulated in fp64 in CSR order.  One warp per atom.
__global__ void k_force_gather(ListView lv, int64_t N, const float* __restrict__ g_list, double* __restrict__ F, int* flags) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  double fx = 0, fy = 0, fz = 0;
  for (int64_t k = lv.rowptr[i] + lane; k < lv.rowptr[i + 1]; k += 32) {
    const int j = (int)(lv.keys[k] >> 24);
    const int64_t kr = lv.rowptr[j] + lv.revpos[k];
    fx += (double)g_list[3 * k] - (double)g_list[3 * kr];
    fy += (double)g_list[3 * k + 1] - (double)g_list[3 * kr + 1];
    fz += (double)g_list[3 * k + 2] - (double)g_list[3 * kr + 2];
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    fx += __shfl_xor_sync(0xffffffffu, fx, d);
    fy += __shfl_xor_sync(0xffffffffu, fy, d);
    fz += __shfl_xor_sync(0xffffffffu, fz, d);
  }
  if (lane == 0) {
    F[3 * i] = fx; F[3 * i + 1] = fy; F[3 * i + 2] = fz;
    if (!(isfinite(fx) && isfinite(fy) && isfinite(fz))) flags[FLAG_NONFINITE] = 1;
  }
}

// Virial W[a][b] = -sum_e (rvec_e)_a (g_e)_b over the list edges (g = 0 on inactive ones); rvec_e in fp64 with
// the expression of the list criterion.  Warps stride over the atoms, lanes over a row; fixed-shape reduction: lane tree,
// warp partials in shared memory, block partials [gridDim.x][9], then k_virial_final (one block) — deterministic, no atomics.
__global__ void __launch_bounds__(256) k_virial_partial(ListView lv, const double* __restrict__ pos, int64_t N, const float* __restrict__ g_list,
                                                        double* __restrict__ partial) {
  __shared__ double sh[8][9];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double w[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  for (int64_t i = (int64_t)blockIdx.x * 8 + warp; i < N; i += (int64_t)gridDim.x * 8) {
    for (int64_t k = lv.rowptr[i] + lane; k < lv.rowptr[i + 1]; k += 32) {
      double d[3]; int j;
      edge_d2(pos, i, lv.keys[k], lv.H, &d[0], &d[1], &d[2], &j);
      const double g[3] = {(double)g_list[3 * k], (double)g_list[3 * k + 1], (double)g_list[3 * k + 2]};
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) w[3 * a + b] -= d[a] * g[b];
    }
  }
#pragma unroll
  for (int q = 0; q < 9; ++q) {
#pragma unroll
    for (int dd = 16; dd > 0; dd >>= 1) w[q] += __shfl_xor_sync(0xffffffffu, w[q], dd);
    if (lane == 0) sh[warp][q] = w[q];
  }
  __syncthreads();
  if (threadIdx.x < 9) {
    double s = 0;
    for (int ww = 0; ww < 8; ++ww) s += sh[ww][threadIdx.x];
    partial[(int64_t)blockIdx.x * 9 + threadIdx.x] = s;
  }
}
__global__ void k_virial_final(const double* __restrict__ partial, int nb, double* __restrict__ W) {
  if (threadIdx.x >= 9) return;
  double s = 0;
  for (int b = 0; b < nb; ++b) s += partial[(int64_t)b * 9 + threadIdx.x];
  W[threadIdx.x] = s;
}

// E = sum_i E_i in fp64: fixed-shape two-stage tree (deterministic)
__global__ void k_energy_partial(const float* __restrict__ e_atom, int64_t N, double* __restrict__ partial) {
  __shared__ double sh[256];
  double s = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) s += (double)e_atom[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int d = 128; d > 0; d >>= 1) {
    if (threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void k_energy_final(const double* __restrict__ partial, int nb, double* __restrict__ E, int* flags) {
  __shared__ double sh[256];
  double s = 0;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) s += partial[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int d = 128; d > 0; d >>= 1) {
    if (threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) { *E = sh[0]; if (!isfinite(sh[0])) flags[FLAG_NONFINITE] = 1; }
}

}  // namespace allegro
