// neighbor.cu — row a-1: device cell-list neighbour builder emitting a sorted CSR edge list.
//
// PAPER.md:93 ("radial cutoff"), north_star item (1); readings A16 (fp64 criterion, expression order),
// A17 (images), A22 (rebuild rule).  Steps: wrap -> bin (histogram, scan, scatter) -> count pass ->
// int64 scan -> fill pass -> per-row rank sort by key (j, sx, sy, sz) -> reverse-edge position.
// An edge is stored as one 64-bit key  j<<24 | (sx+128)<<16 | (sy+128)<<8 | (sz+128).
// Every kernel can run "conditionally": it returns at once when flags[FLAG_REBUILD] == 0, so that the MD
// loop can enqueue a rebuild without a host round trip.
#include <algorithm>
#include <cmath>
#include <cstdio>

#include "model.h"

namespace allegro {
namespace {

constexpr int SCAN_T = 1024;

__global__ void k_scan_block(const int* __restrict__ cnt, const int64_t* __restrict__ in64, int64_t* __restrict__ out,
                             int64_t* __restrict__ block_sum, int64_t n, const int* flag) {
  if (flag && *flag == 0) return;
  __shared__ int64_t warp_tot[32];
  int64_t i = (int64_t)blockIdx.x * SCAN_T + threadIdx.x;
  int64_t v = 0;
  if (i < n) v = cnt ? (int64_t)cnt[i] : in64[i];
  int64_t x = v;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int64_t y = __shfl_up_sync(0xffffffffu, x, d);
    if (lane >= d) x += y;
  }
  if (lane == 31) warp_tot[wid] = x;
  __syncthreads();
  if (wid == 0) {
    int64_t t = warp_tot[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      int64_t y = __shfl_up_sync(0xffffffffu, t, d);
      if (lane >= d) t += y;
    }
    warp_tot[lane] = t;
  }
  __syncthreads();
  int64_t base = wid ? warp_tot[wid - 1] : 0;
  if (i < n) out[i] = base + x - v;  // exclusive
  if (threadIdx.x == SCAN_T - 1) block_sum[blockIdx.x] = base + x;
}

__global__ void k_scan_add(int64_t* __restrict__ out, const int64_t* __restrict__ block_off, int64_t n,
                           const int64_t* __restrict__ total, const int* flag) {
  if (flag && *flag == 0) return;
  int64_t i = (int64_t)blockIdx.x * SCAN_T + threadIdx.x;
  if (i < n) out[i] += block_off[blockIdx.x];
  else if (i == n && total) out[n] = *total;
}

// small inputs: one block walks the array in slices of SCAN_T with a running carry (one launch instead of five)
__global__ void __launch_bounds__(SCAN_T) k_scan_small(const int* __restrict__ cnt, int64_t* __restrict__ out, int64_t n, const int* flag) {
  if (flag && *flag == 0) return;
  __shared__ int64_t warp_tot[32];
  __shared__ int64_t carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int64_t i0 = 0; i0 < n; i0 += SCAN_T) {
    const int64_t i = i0 + threadIdx.x;
    const int64_t v = (i < n) ? (int64_t)cnt[i] : 0;
    int64_t x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int64_t y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) warp_tot[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int64_t t = warp_tot[lane];
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int64_t y = __shfl_up_sync(0xffffffffu, t, d);
        if (lane >= d) t += y;
      }
      warp_tot[lane] = t;
    }
    __syncthreads();
    const int64_t carry = carry_s;
    const int64_t base = carry + (wid ? warp_tot[wid - 1] : 0);
    if (i < n) out[i] = base + x - v;
    __syncthreads();
    if (threadIdx.x == SCAN_T - 1) carry_s = base + x;
    __syncthreads();
  }
  if (threadIdx.x == 0) out[n] = carry_s;
}

}  // namespace

// out[0..n] = exclusive scan of cnt[0..n-1] (out[n] = total).  Three levels of 1024 (n <= 2^30).
int scan_counts(Model* m, const int* cnt, int64_t* out, int64_t n, DevBuf* tmp, const int* flag, cudaStream_t st) {
  if (n <= 0) {
    cudaMemsetAsync(out, 0, sizeof(int64_t), st);
    return 0;
  }
  if (n <= 16 * SCAN_T) {
    k_scan_small<<<1, SCAN_T, 0, st>>>(cnt, out, n, flag);
    m->launches += 1;
    return 0;
  }
  const int64_t nb1 = (n + SCAN_T - 1) / SCAN_T, nb2 = (nb1 + SCAN_T - 1) / SCAN_T, nb3 = (nb2 + SCAN_T - 1) / SCAN_T;
  if (nb3 > 1) { m->err = "scan: n too large"; return ALLEGRO_ERR_UNSUPPORTED; }
  if (int rc = ensure(m, tmp, sizeof(int64_t) * (2 * nb1 + 2 * nb2 + 8))) return rc;
  int64_t* s1 = tmp->as<int64_t>();      // level-1 block totals [nb1]
  int64_t* o1 = s1 + nb1;                // their exclusive scan  [nb1]
  int64_t* s2 = o1 + nb1;                // level-2 block totals [nb2]
  int64_t* o2 = s2 + nb2;                // their exclusive scan  [nb2]
  int64_t* s3 = o2 + nb2;                // grand total [1]
  k_scan_block<<<(unsigned)nb1, SCAN_T, 0, st>>>(cnt, nullptr, out, s1, n, flag);
  k_scan_block<<<(unsigned)nb2, SCAN_T, 0, st>>>(nullptr, s1, o1, s2, nb1, flag);
  k_scan_block<<<1, SCAN_T, 0, st>>>(nullptr, s2, o2, s3, nb2, flag);
  k_scan_add<<<(unsigned)nb2, SCAN_T, 0, st>>>(o1, o2, nb1, nullptr, flag);
  k_scan_add<<<(unsigned)((n + 1 + SCAN_T - 1) / SCAN_T), SCAN_T, 0, st>>>(out, o1, n, s3, flag);
  m->launches += 5;
  return 0;
}

namespace {

__device__ __forceinline__ uint64_t make_key(int j, int sx, int sy, int sz) {
  return ((uint64_t)(uint32_t)j << 24) | ((uint64_t)(sx + 128) << 16) | ((uint64_t)(sy + 128) << 8) | (uint64_t)(sz + 128);
}

// as image_shift of edge_kernels.cuh (the two must stay the same expression)
__device__ __forceinline__ double nl_image_shift(const double* H, int c, int sx, int sy, int sz) {
  return __dadd_rn(__dadd_rn(__dmul_rn((double)sx, H[c]), __dmul_rn((double)sy, H[3 + c])), __dmul_rn((double)sz, H[6 + c]));
}

struct Grid {
  double H[9], Hinv[9];    // cell (rows = lattice vectors) and its inverse: fractional coordinates f = x Hinv
  double h[3];             // orthorhombic cell: bin width per axis
  int nc[3];
  int ortho;
};

__global__ void k_bin_count(const double* __restrict__ pos, int64_t N, Grid g, int* __restrict__ img, int* __restrict__ cell_of,
                            int* __restrict__ cell_cnt, const int* flags) {
  if (flags[FLAG_REBUILD] == 0) return;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int c[3];
  if (g.ortho) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double x = pos[3 * i + d];
      double w = floor(x / g.H[4 * d]);
      double xt = x - w * g.H[4 * d];
      int ci = (int)(xt / g.h[d]);
      ci = max(0, min(ci, g.nc[d] - 1));
      c[d] = ci;
      img[3 * i + d] = (int)w;
    }
  } else {
    // general cell (A27): bins in fractional coordinates; every point within R of x has |delta f_d| <= R / width_d <= 1 / nc_d
    const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double f = x * g.Hinv[d] + y * g.Hinv[3 + d] + z * g.Hinv[6 + d];
      const double w = floor(f);
      int ci = (int)((f - w) * (double)g.nc[d]);
      ci = max(0, min(ci, g.nc[d] - 1));
      c[d] = ci;
      img[3 * i + d] = (int)w;
    }
  }
  int cid = (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
  cell_of[i] = cid;
  atomicAdd(&cell_cnt[cid], 1);
}

__global__ void k_bin_scatter(int64_t N, const int* __restrict__ cell_of, const int64_t* __restrict__ cell_start,
                              int* __restrict__ cell_fill, int* __restrict__ sorted, const int* flags) {
  if (flags[FLAG_REBUILD] == 0) return;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int cid = cell_of[i];
  int slot = atomicAdd(&cell_fill[cid], 1);
  sorted[cell_start[cid] + slot] = (int)i;
}

// One warp per centre atom.  MODE 0: count; MODE 1: fill unsorted keys at rowptr[i].
template <int MODE>
__global__ void k_nbr_pass(const double* __restrict__ pos, int64_t N, Grid g, double R2, const int* __restrict__ img,
                           const int* __restrict__ cell_of, const int64_t* __restrict__ cell_start,
                           const int* __restrict__ sorted, int* __restrict__ row_cnt, const int64_t* __restrict__ rowptr,
                           uint64_t* __restrict__ keys_tmp, int64_t cap, int* flags) {
  if (flags[FLAG_REBUILD] == 0) return;
  const int lane = threadIdx.x & 31;
  int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
  const int wix = img[3 * i], wiy = img[3 * i + 1], wiz = img[3 * i + 2];
  int cid = cell_of[i];
  const int cz = cid % g.nc[2], cy = (cid / g.nc[2]) % g.nc[1], cx = cid / (g.nc[2] * g.nc[1]);
  int64_t base = MODE ? rowptr[i] : 0;
  int total = 0;
  for (int ox = -1; ox <= 1; ++ox)
    for (int oy = -1; oy <= 1; ++oy)
      for (int oz = -1; oz <= 1; ++oz) {
        int nx = cx + ox, ny = cy + oy, nz = cz + oz;
        int ix = (nx < 0) ? -1 : (nx >= g.nc[0] ? 1 : 0);
        int iy = (ny < 0) ? -1 : (ny >= g.nc[1] ? 1 : 0);
        int iz = (nz < 0) ? -1 : (nz >= g.nc[2] ? 1 : 0);
        nx -= ix * g.nc[0]; ny -= iy * g.nc[1]; nz -= iz * g.nc[2];
        int ncid = (nx * g.nc[1] + ny) * g.nc[2] + nz;
        int64_t b = cell_start[ncid], e = cell_start[ncid + 1];
        for (int64_t k0 = b; k0 < e; k0 += 32) {
          int64_t k = k0 + lane;
          bool ok = false;
          int j = 0, sx = 0, sy = 0, sz = 0;
          if (k < e) {
            j = sorted[k];
            sx = ix + wix - img[3 * j]; sy = iy + wiy - img[3 * j + 1]; sz = iz + wiz - img[3 * j + 2];
            // A16 / A27: dx = (x_j - x_i) + (s_1 a_1x + s_2 a_2x + s_3 a_3x), d2 = dx*dx + dy*dy + dz*dz, all fp64, no FMA contraction
            double dx = __dadd_rn(__dsub_rn(pos[3 * j], xi), nl_image_shift(g.H, 0, sx, sy, sz));
            double dy = __dadd_rn(__dsub_rn(pos[3 * j + 1], yi), nl_image_shift(g.H, 1, sx, sy, sz));
            double dz = __dadd_rn(__dsub_rn(pos[3 * j + 2], zi), nl_image_shift(g.H, 2, sx, sy, sz));
            double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            ok = (d2 < R2) && !(j == (int)i && sx == 0 && sy == 0 && sz == 0);
          }
          unsigned bal = __ballot_sync(0xffffffffu, ok);
          if (MODE == 1 && ok) {
            if (sx < -128 || sx > 127 || sy < -128 || sy > 127 || sz < -128 || sz > 127) atomicExch(&flags[FLAG_ERR_SHIFT], 1);
            int64_t dst = base + total + __popc(bal & ((1u << lane) - 1u));
            if (dst < cap) keys_tmp[dst] = make_key(j, sx, sy, sz);
          }
          total += __popc(bal);
        }
      }
  if (MODE == 0 && lane == 0) row_cnt[i] = total;
}

// The new row offsets are scanned into a scratch array: when the rebuilt list would not fit, the old list (offsets included)
// stays intact, the rebuild is cancelled and the integrator is halted (FLAG_HALT); the host regrows and finishes the call.
__global__ void k_check_cap(const int64_t* rowptr_new, int64_t N, int64_t cap, int* flags) {
  if (flags[FLAG_REBUILD] == 0) return;
  if (rowptr_new[N] > cap) { flags[FLAG_ERR_CAP] = 1; flags[FLAG_HALT] = 1; flags[FLAG_REBUILD] = 0; }
}
__global__ void k_commit_rowptr(const int64_t* __restrict__ rowptr_new, int64_t* __restrict__ rowptr, int64_t N, const int* flags) {
  if (flags[FLAG_REBUILD] == 0) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= N) rowptr[i] = rowptr_new[i];
}

// One warp per row: rank of each key among the row's keys (keys are distinct) -> sorted position.
__global__ void k_row_sort(int64_t N, const int64_t* __restrict__ rowptr, const uint64_t* __restrict__ keys_tmp,
                           uint64_t* __restrict__ keys, int64_t cap, const int* flags) {
  if (flags[FLAG_REBUILD] == 0 || flags[FLAG_ERR_CAP]) return;
  const int lane = threadIdx.x & 31;
  int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const int64_t b = rowptr[i], e = rowptr[i + 1];
  for (int64_t k = b + lane; k < e; k += 32) {
    const uint64_t key = keys_tmp[k];
    int rank = 0;
    for (int64_t q = b; q < e; ++q) rank += (keys_tmp[q] < key);
    keys[b + rank] = key;
  }
}

// revpos[e] = position inside row j of the reverse edge (j -> i, -s): binary search in the sorted row.
__global__ void k_reverse(int64_t N, const int64_t* __restrict__ rowptr, const uint64_t* __restrict__ keys,
                          int* __restrict__ revpos, int* flags) {
  if (flags[FLAG_REBUILD] == 0 || flags[FLAG_ERR_CAP]) return;
  const int lane = threadIdx.x & 31;
  int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= N) return;
  const int64_t b = rowptr[i], e = rowptr[i + 1];
  for (int64_t k = b + lane; k < e; k += 32) {
    const uint64_t key = keys[k];
    const int j = (int)(key >> 24);
    const int sx = (int)((key >> 16) & 255) - 128, sy = (int)((key >> 8) & 255) - 128, sz = (int)(key & 255) - 128;
    const uint64_t want = make_key((int)i, -sx, -sy, -sz);
    int64_t lo = rowptr[j], hi = rowptr[j + 1];
    const int64_t jb = lo;
    while (lo < hi) {
      int64_t mid = (lo + hi) >> 1;
      if (keys[mid] < want) lo = mid + 1; else hi = mid;
    }
    if (lo >= rowptr[j + 1] || keys[lo] != want) atomicExch(&flags[FLAG_ERR_SHIFT], 2);  // asymmetric list: cannot happen
    revpos[k] = (int)(lo - jb);
  }
}

__global__ void k_finish_build(const double* __restrict__ pos, double* __restrict__ r_build, int64_t n3, int* flags) {
  if (flags[FLAG_REBUILD] == 0) return;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n3) r_build[i] = pos[i];
  if (i == 0) flags[FLAG_NREBUILD] += 1;
}

__global__ void k_export(int64_t E, const uint64_t* __restrict__ keys, int32_t* __restrict__ col, int8_t* __restrict__ shift) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= E) return;
  uint64_t key = keys[k];
  if (col) col[k] = (int32_t)(key >> 24);
  if (shift) {
    shift[3 * k] = (int8_t)((int)((key >> 16) & 255) - 128);
    shift[3 * k + 1] = (int8_t)((int)((key >> 8) & 255) - 128);
    shift[3 * k + 2] = (int8_t)((int)(key & 255) - 128);
  }
}

}  // namespace

// conditional == false: flags[FLAG_REBUILD] is set here, the list is sized exactly (one host sync after the
// count pass) and buffers are (re)allocated.  conditional == true: every kernel checks the device flag, buffers
// keep their capacity, overflow raises FLAG_ERR_CAP (reported by the caller after its final sync).
int nl_build(Model* m, const double* pos, int64_t N, const double* cell, double cutoff, double skin, bool conditional,
             cudaStream_t st) {
  NeighborList& nl = m->nl;
  int* flags = m->flags.as<int>();
  const double R = cutoff + skin;
  if (!conditional) {
    // cell: rows = lattice vectors (A27).  Perpendicular widths w_d = 1 / |column d of H^-1| (= L_d for an orthorhombic box)
    nl.ortho = true;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        nl.H[3 * a + b] = cell[3 * a + b];
        if (a != b && cell[3 * a + b] != 0.0) nl.ortho = false;
      }
    const double* H = nl.H;
    const double det = H[0] * (H[4] * H[8] - H[5] * H[7]) - H[1] * (H[3] * H[8] - H[5] * H[6]) + H[2] * (H[3] * H[7] - H[4] * H[6]);
    if (!(det > 0.0) || !std::isfinite(det)) { m->err = "cell must be right-handed with positive volume (cell lengths must be positive)"; return ALLEGRO_ERR_INVALID; }
    const double cof[9] = {H[4] * H[8] - H[5] * H[7], H[2] * H[7] - H[1] * H[8], H[1] * H[5] - H[2] * H[4],
                           H[5] * H[6] - H[3] * H[8], H[0] * H[8] - H[2] * H[6], H[2] * H[3] - H[0] * H[5],
                           H[3] * H[7] - H[4] * H[6], H[1] * H[6] - H[0] * H[7], H[0] * H[4] - H[1] * H[3]};
    for (int k = 0; k < 9; ++k) nl.Hinv[k] = cof[k] / det;
    for (int d = 0; d < 3; ++d) {
      const double width = nl.ortho ? H[4 * d]
                                    : 1.0 / std::sqrt(nl.Hinv[d] * nl.Hinv[d] + nl.Hinv[3 + d] * nl.Hinv[3 + d] + nl.Hinv[6 + d] * nl.Hinv[6 + d]);
      if (!(width > 0.0)) { m->err = "cell lengths must be positive"; return ALLEGRO_ERR_INVALID; }
      if (R > width) { m->err = "r_cut + skin exceeds the smallest box length (perpendicular width of the cell; A17)"; return ALLEGRO_ERR_CUTOFF; }
      int64_t c = (int64_t)floor(width / (R * (1.0 + 1e-9)));
      nl.nc[d] = (int)std::max<int64_t>(1, std::min<int64_t>(c, 1024));
    }
    // keep the number of cells bounded by ~N (tiny systems in huge boxes)
    while ((int64_t)nl.nc[0] * nl.nc[1] * nl.nc[2] > std::max<int64_t>(64, 4 * N)) {
      int d = (nl.nc[0] >= nl.nc[1] && nl.nc[0] >= nl.nc[2]) ? 0 : (nl.nc[1] >= nl.nc[2] ? 1 : 2);
      nl.nc[d] = (nl.nc[d] + 1) / 2;
    }
    nl.N = N; nl.cutoff = cutoff; nl.skin = skin; nl.valid = false;
    const int64_t ncell = (int64_t)nl.nc[0] * nl.nc[1] * nl.nc[2];
    int rc = 0;
    rc |= ensure(m, &nl.r_build, sizeof(double) * 3 * N + 8);
    rc |= ensure(m, &nl.img, sizeof(int) * 3 * N + 8);
    rc |= ensure(m, &nl.cell_of, sizeof(int) * N + 8);
    rc |= ensure(m, &nl.cell_cnt, sizeof(int) * ncell);
    rc |= ensure(m, &nl.cell_fill, sizeof(int) * ncell);
    rc |= ensure(m, &nl.cell_start, sizeof(int64_t) * (ncell + 1));
    rc |= ensure(m, &nl.sorted, sizeof(int) * N + 8);
    rc |= ensure(m, &nl.row_cnt, sizeof(int) * N + 8);
    rc |= ensure(m, &nl.rowptr, sizeof(int64_t) * (N + 1));
    rc |= ensure(m, &nl.rowptr_new, sizeof(int64_t) * (N + 1));
    if (rc) return ALLEGRO_ERR_ALLOC;
    int one = 1;
    cudaMemcpyAsync(&flags[FLAG_REBUILD], &one, sizeof(int), cudaMemcpyHostToDevice, st);
  }
  const int64_t ncell = (int64_t)nl.nc[0] * nl.nc[1] * nl.nc[2];
  Grid g;
  for (int k = 0; k < 9; ++k) { g.H[k] = nl.H[k]; g.Hinv[k] = nl.Hinv[k]; }
  for (int d = 0; d < 3; ++d) { g.nc[d] = nl.nc[d]; g.h[d] = nl.H[4 * d] / nl.nc[d]; }
  g.ortho = nl.ortho ? 1 : 0;
  const int T = 256;
  const unsigned gridN = (unsigned)((N + T - 1) / T), gridW = (unsigned)((N * 32 + T - 1) / T);
  if (N == 0) {
    nl.E_list = 0; nl.valid = true;
    cudaMemsetAsync(nl.rowptr.p, 0, sizeof(int64_t), st);
    cudaMemsetAsync(&flags[FLAG_REBUILD], 0, sizeof(int), st);
    return 0;
  }
  // (conditional) zero of the histograms: cheap, done unconditionally
  cudaMemsetAsync(nl.cell_cnt.p, 0, sizeof(int) * ncell, st);
  cudaMemsetAsync(nl.cell_fill.p, 0, sizeof(int) * ncell, st);
  k_bin_count<<<gridN, T, 0, st>>>(pos, N, g, nl.img.as<int>(), nl.cell_of.as<int>(), nl.cell_cnt.as<int>(), flags);
  if (int rc = scan_counts(m, nl.cell_cnt.as<int>(), nl.cell_start.as<int64_t>(), ncell, &nl.scan_tmp, &flags[FLAG_REBUILD], st)) return rc;
  k_bin_scatter<<<gridN, T, 0, st>>>(N, nl.cell_of.as<int>(), nl.cell_start.as<int64_t>(), nl.cell_fill.as<int>(), nl.sorted.as<int>(), flags);
  k_nbr_pass<0><<<gridW, T, 0, st>>>(pos, N, g, R * R, nl.img.as<int>(), nl.cell_of.as<int>(), nl.cell_start.as<int64_t>(),
                                     nl.sorted.as<int>(), nl.row_cnt.as<int>(), nullptr, nullptr, 0, flags);
  if (int rc = scan_counts(m, nl.row_cnt.as<int>(), nl.rowptr_new.as<int64_t>(), N, &nl.scan_tmp, &flags[FLAG_REBUILD], st)) return rc;
  m->launches += 3;
  if (!conditional) {
    int64_t E = 0;
    cudaMemcpyAsync(&E, nl.rowptr_new.as<int64_t>() + N, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(m, e, "neighbor count pass");
    nl.E_list = E;
    int64_t cap = E + (int64_t)(nl.slack_frac * (double)E) + nl.slack_extra;   // slack for the conditional rebuilds of the MD loop
    int rc = 0;
    rc |= ensure(m, &nl.keys_tmp, sizeof(uint64_t) * cap);
    rc |= ensure(m, &nl.keys, sizeof(uint64_t) * cap);
    rc |= ensure(m, &nl.revpos, sizeof(int) * cap);
    rc |= ensure(m, &m->g_list, sizeof(float) * 3 * cap);
    if (rc) return ALLEGRO_ERR_ALLOC;
    nl.cap = std::min<int64_t>({(int64_t)(nl.keys.bytes / 8), (int64_t)(nl.keys_tmp.bytes / 8), (int64_t)(nl.revpos.bytes / 4),
                                (int64_t)(m->g_list.bytes / 12)});
  }
  k_check_cap<<<1, 1, 0, st>>>(nl.rowptr_new.as<int64_t>(), N, nl.cap, flags);
  k_commit_rowptr<<<(unsigned)((N + 1 + T - 1) / T), T, 0, st>>>(nl.rowptr_new.as<int64_t>(), nl.rowptr.as<int64_t>(), N, flags);
  k_nbr_pass<1><<<gridW, T, 0, st>>>(pos, N, g, R * R, nl.img.as<int>(), nl.cell_of.as<int>(), nl.cell_start.as<int64_t>(),
                                     nl.sorted.as<int>(), nullptr, nl.rowptr.as<int64_t>(), nl.keys_tmp.as<uint64_t>(), nl.cap, flags);
  k_row_sort<<<gridW, T, 0, st>>>(N, nl.rowptr.as<int64_t>(), nl.keys_tmp.as<uint64_t>(), nl.keys.as<uint64_t>(), nl.cap, flags);
  k_reverse<<<gridW, T, 0, st>>>(N, nl.rowptr.as<int64_t>(), nl.keys.as<uint64_t>(), nl.revpos.as<int>(), flags);
  k_finish_build<<<(unsigned)((3 * N + T - 1) / T), T, 0, st>>>(pos, nl.r_build.as<double>(), 3 * N, flags);
  m->launches += 5;
  if (!conditional) {
    int zero = 0;
    cudaMemcpyAsync(&flags[FLAG_REBUILD], &zero, sizeof(int), cudaMemcpyHostToDevice, st);
    nl.valid = true;
  }
  return 0;
}

int nl_export(Model* m, int64_t* rowptr, int32_t* col, int8_t* shift, cudaStream_t st) {
  NeighborList& nl = m->nl;
  if (rowptr) cudaMemcpyAsync(rowptr, nl.rowptr.p, sizeof(int64_t) * (nl.N + 1), cudaMemcpyDeviceToDevice, st);
  if ((col || shift) && nl.E_list > 0)
    k_export<<<(unsigned)((nl.E_list + 255) / 256), 256, 0, st>>>(nl.E_list, nl.keys.as<uint64_t>(), col, shift);
  return 0;
}

}  // namespace allegro
