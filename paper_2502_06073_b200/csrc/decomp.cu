// decomp.cu — SURVEY.md 8f-3 / 8e: spatial decomposition of the strictly local model ("strictly-local", the property
// behind the paper's 0.964 parallel efficiency on Aurora).  One rank owns the atoms of a brick of the orthorhombic cell and
// evaluates E_i for those; it needs every atom within r_halo of the brick as a ghost (neighbour only).  Design for one NVSwitch
// node: coordinates are replicated on every rank (24 B per atom, negligible beside the force evaluation), so the ghost selection
// is a local compaction — no position exchange — and the only collective of a step is one all-reduce of the force array (ghost
// forces land on their owners there) plus the 8-byte energy.  The kernels here: brick selection (owned first, then ghost images,
// both in ascending atom order: deterministic), the conflict-free scatter of the local forces back to global atom order, and the
// velocity-Verlet half-steps on caller arrays (every rank integrates the replicated state identically).
#include <algorithm>

#include "model.h"

namespace allegro {
namespace {

struct Brick {
  double L[3], lo[3], hi[3], origin[3];   // cell lengths; brick bounds (decomposed dims); local = wrapped + s L - origin
  int dec[3];                              // 1 = dimension is decomposed (local box is not periodic there)
  double halo;
};

__device__ __forceinline__ double wrap_d(double x, double L) { return x - floor(x / L) * L; }

// MODE 0: per atom, owned flag and number of ghost images.  MODE 1: fill.
template <int MODE>
__global__ void k_decomp_select(const double* __restrict__ pos, int64_t N, Brick b, int* __restrict__ own_cnt, int* __restrict__ gh_cnt,
                                const int64_t* __restrict__ own_off, const int64_t* __restrict__ gh_off, int64_t n_owned, int64_t cap,
                                double* __restrict__ lpos, int64_t* __restrict__ lsrc) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  double w[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) w[d] = b.dec[d] ? wrap_d(pos[3 * i + d], b.L[d]) : pos[3 * i + d];
  bool owned = true;
#pragma unroll
  for (int d = 0; d < 3; ++d)
    if (b.dec[d]) owned = owned && (w[d] >= b.lo[d] && w[d] < b.hi[d]);
  int ng = 0;
  int64_t gdst = MODE ? n_owned + gh_off[i] : 0;
  for (int sx = -b.dec[0]; sx <= b.dec[0]; ++sx)
    for (int sy = -b.dec[1]; sy <= b.dec[1]; ++sy)
      for (int sz = -b.dec[2]; sz <= b.dec[2]; ++sz) {
        if (owned && sx == 0 && sy == 0 && sz == 0) continue;
        const double c[3] = {w[0] + sx * b.L[0], w[1] + sy * b.L[1], w[2] + sz * b.L[2]};
        bool in = true;
#pragma unroll
        for (int d = 0; d < 3; ++d)
          if (b.dec[d]) in = in && (c[d] >= b.lo[d] - b.halo && c[d] < b.hi[d] + b.halo);
        if (!in) continue;
        if (MODE == 1 && gdst < cap) {
          lpos[3 * gdst] = c[0] - b.origin[0]; lpos[3 * gdst + 1] = c[1] - b.origin[1]; lpos[3 * gdst + 2] = c[2] - b.origin[2];
          lsrc[gdst] = i;
        }
        ++gdst; ++ng;
      }
  if (MODE == 0) { own_cnt[i] = owned ? 1 : 0; gh_cnt[i] = ng; }
  if (MODE == 1 && owned) {
    const int64_t dst = own_off[i];
    if (dst < cap) {
      lpos[3 * dst] = w[0] - b.origin[0]; lpos[3 * dst + 1] = w[1] - b.origin[1]; lpos[3 * dst + 2] = w[2] - b.origin[2];
      lsrc[dst] = i;
    }
  }
}

__global__ void k_decomp_gather_species(const int64_t* __restrict__ lsrc, int64_t n, const int32_t* __restrict__ species, int32_t* __restrict__ lspecies) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) lspecies[k] = species[lsrc[k]];
}

// every global atom appears at most once in a rank's local set (brick + 2 halo <= L is checked on the host): plain stores
__global__ void k_decomp_scatter(const double* __restrict__ F_local, const int64_t* __restrict__ lsrc, int64_t n, double* __restrict__ F_global) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int64_t i = lsrc[k];
  F_global[3 * i] = F_local[3 * k]; F_global[3 * i + 1] = F_local[3 * k + 1]; F_global[3 * i + 2] = F_local[3 * k + 2];
}

constexpr double ACC_CONV_D = 9.648533212e-3;
__global__ void k_kick_drift_ext(double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ F, const double* __restrict__ mass,
                                 int64_t N, double dt, int drift) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 3 * N) return;
  const double v = vel[idx] + 0.5 * dt * ACC_CONV_D * F[idx] / mass[idx / 3];
  vel[idx] = v;
  if (drift) pos[idx] += dt * v;
}

}  // namespace

int decomp_select(Model* m, const double* pos, const int32_t* species, int64_t N, const double* cell, const int32_t* grid, const int32_t* coord,
                  double r_halo, int64_t cap, double* lpos, int32_t* lspecies, int64_t* lsrc, int64_t* counts_host, double* local_cell_host,
                  cudaStream_t st) {
  Brick b;
  b.halo = r_halo;
  for (int d = 0; d < 3; ++d) {
    for (int e = 0; e < 3; ++e)
      if (d != e && cell[3 * d + e] != 0.0) { m->err = "decomposition needs an orthorhombic cell"; return ALLEGRO_ERR_UNSUPPORTED; }
    b.L[d] = cell[4 * d];
    if (grid[d] < 1 || coord[d] < 0 || coord[d] >= grid[d]) { m->err = "bad rank grid"; return ALLEGRO_ERR_INVALID; }
    b.dec[d] = grid[d] > 1 ? 1 : 0;
    const double w = b.L[d] / grid[d];
    b.lo[d] = w * coord[d];
    b.hi[d] = (coord[d] + 1 == grid[d]) ? b.L[d] : w * (coord[d] + 1);
    if (b.dec[d] && (b.hi[d] - b.lo[d]) + 2.0 * r_halo > b.L[d]) {
      m->err = "brick + 2 halo exceeds the box length: an atom would appear twice in a rank's local set";
      return ALLEGRO_ERR_UNSUPPORTED;
    }
    // local coordinates start at 0; the local box is padded by one more halo so that no pair forms across its periodic wrap
    b.origin[d] = b.dec[d] ? b.lo[d] - r_halo : 0.0;
    for (int e = 0; e < 3; ++e) local_cell_host[3 * d + e] = 0.0;
    local_cell_host[4 * d] = b.dec[d] ? (b.hi[d] - b.lo[d]) + 3.0 * r_halo + 1.0 : b.L[d];
  }
  DevBuf& tmp = m->decomp_tmp;
  if (int rc = ensure(m, &tmp, (sizeof(int) * 2 + sizeof(int64_t) * 2) * (size_t)(N + 2) + 64)) return rc;
  int* own_cnt = tmp.as<int>();
  int* gh_cnt = own_cnt + (N + 2);
  int64_t* own_off = reinterpret_cast<int64_t*>(gh_cnt + (N + 2));
  int64_t* gh_off = own_off + (N + 2);
  const int T = 256;
  const unsigned g = (unsigned)((N + T - 1) / T);
  if (N > 0) k_decomp_select<0><<<g, T, 0, st>>>(pos, N, b, own_cnt, gh_cnt, nullptr, nullptr, 0, 0, nullptr, nullptr);
  if (int rc = scan_counts(m, own_cnt, own_off, N, &m->nl.scan_tmp, nullptr, st)) return rc;
  if (int rc = scan_counts(m, gh_cnt, gh_off, N, &m->nl.scan_tmp, nullptr, st)) return rc;
  int64_t tot[2] = {0, 0};
  cudaMemcpyAsync(&tot[0], own_off + N, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
  cudaMemcpyAsync(&tot[1], gh_off + N, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
  cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_decomp_select");
  counts_host[0] = tot[0]; counts_host[1] = tot[0] + tot[1];
  if (counts_host[1] > cap) { m->err = "local atom capacity too small"; return ALLEGRO_ERR_ALLOC; }
  if (N > 0) {
    k_decomp_select<1><<<g, T, 0, st>>>(pos, N, b, nullptr, nullptr, own_off, gh_off, tot[0], cap, lpos, lsrc);
    if (counts_host[1] > 0 && lspecies)
      k_decomp_gather_species<<<(unsigned)((counts_host[1] + T - 1) / T), T, 0, st>>>(lsrc, counts_host[1], species, lspecies);
  }
  return 0;
}

int decomp_scatter(const double* F_local, const int64_t* lsrc, int64_t n_local, double* F_global, int64_t N, cudaStream_t st) {
  cudaMemsetAsync(F_global, 0, sizeof(double) * 3 * (size_t)N, st);
  if (n_local > 0) k_decomp_scatter<<<(unsigned)((n_local + 255) / 256), 256, 0, st>>>(F_local, lsrc, n_local, F_global);
  return 0;
}

int ext_kick_drift(double* pos, double* vel, const double* F, const double* mass, int64_t N, double dt, int drift, cudaStream_t st) {
  if (N > 0) k_kick_drift_ext<<<(unsigned)((3 * N + 255) / 256), 256, 0, st>>>(pos, vel, F, mass, N, dt, drift);
  return 0;
}

}  // namespace allegro
