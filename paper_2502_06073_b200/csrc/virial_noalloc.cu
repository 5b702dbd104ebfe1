// virial_noalloc.cu — allegro_virial_noalloc: the virial W = -sum_e rvec_e (x) dE/d rvec_e (R5) for callers
// that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  allegro_virial
// (api.cu / network.cu) keeps its block partials in a cudaMalloc'ed buffer of the handle; this variant keeps them in a file-scope
// __device__ array of fixed size, so the call contains no cudaMalloc / cudaFree / allocating library routine and no stream
// synchronisation: two kernel launches on the caller's stream, nothing else.
//
// Limits that follow from the fixed array:
//   * N <= ALLEGRO_VIRIAL_NOALLOC_MAX_ATOMS (1,048,576): one block partial per 256 atoms, 4,096 partials of 9 doubles = 288 KB,
//     held by every GPU that loads the library until the process exits.  Larger systems get ALLEGRO_ERR_UNSUPPORTED.
//   * every call on a device shares the one array: calls that overlap on the GPU (different streams, different handles) race.
//     Calls on one stream are ordered and safe.
//   * the array keeps the last call's contents; nothing has to start at zero here (every partial that the final kernel reads is
//     overwritten by the first kernel of the same call), so no clearing pass is needed.
#include <mutex>

#include "model.h"

namespace allegro {
namespace {

constexpr int VN_ATOMS_PER_BLOCK = 256;                 // 8 warps x 32 atoms
constexpr int VN_MAX_BLOCKS = 4096;
constexpr int64_t VN_MAX_ATOMS = (int64_t)VN_ATOMS_PER_BLOCK * VN_MAX_BLOCKS;
static_assert(VN_MAX_ATOMS == ALLEGRO_VIRIAL_NOALLOC_MAX_ATOMS, "include/allegro.h states the limit");

// In host code this name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress (scratch_for_device below).
static __device__ __align__(256) double g_virial_scratch[(size_t)VN_MAX_BLOCKS * 9];

// list key: j << 24 | (sx + 128) << 16 | (sy + 128) << 8 | (sz + 128)
struct VnCell { double H[9]; };   // rows = lattice vectors

__device__ __forceinline__ void vn_edge(const double* __restrict__ pos, int64_t i, uint64_t key, const VnCell& cl, double* d) {
  const int64_t j = (int64_t)(key >> 24);
  const double sx = (double)((int)((key >> 16) & 255) - 128), sy = (double)((int)((key >> 8) & 255) - 128), sz = (double)((int)(key & 255) - 128);
  // A16 / A27: the expression of the list criterion, fp64, no FMA contraction
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double sh = __dadd_rn(__dadd_rn(__dmul_rn(sx, cl.H[c]), __dmul_rn(sy, cl.H[3 + c])), __dmul_rn(sz, cl.H[6 + c]));
    d[c] = __dadd_rn(__dsub_rn(pos[3 * j + c], pos[3 * i + c]), sh);
  }
}

// Block b covers atoms [256 b, 256 b + 256): warp w the 32 atoms from 256 b + 32 w, lanes stride over a list row.  Fixed-shape
// fp64 reduction (lane tree, warp partials in shared memory, one block partial [9]): deterministic, no atomics.
__global__ void __launch_bounds__(256) k_virial_partial_na(const int64_t* __restrict__ rowptr, const uint64_t* __restrict__ keys,
                                                           const float* __restrict__ g_list, const double* __restrict__ pos, int64_t N,
                                                           VnCell cl, double* __restrict__ partial) {
  __shared__ double sh[8][9];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double w[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  const int64_t i0 = (int64_t)blockIdx.x * VN_ATOMS_PER_BLOCK + warp * 32;
  const int64_t i1 = i0 + 32 < N ? i0 + 32 : N;
  for (int64_t i = i0; i < i1; ++i) {
    for (int64_t k = rowptr[i] + lane; k < rowptr[i + 1]; k += 32) {
      double d[3];
      vn_edge(pos, i, keys[k], cl, d);
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

// one block of 9 warps: warp q sums component q over the nb block partials (lanes stride, then a lane tree)
__global__ void __launch_bounds__(288) k_virial_final_na(const double* __restrict__ partial, int nb, double* __restrict__ W) {
  const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;
  double s = 0;
  for (int b = lane; b < nb; b += 32) s += partial[(int64_t)b * 9 + q];
#pragma unroll
  for (int dd = 16; dd > 0; dd >>= 1) s += __shfl_xor_sync(0xffffffffu, s, dd);
  if (lane == 0) W[q] = s;
}

// Device address of the scratch array, looked up once per device with that device current.
constexpr int VN_MAX_DEVICES = 64;
std::mutex g_vn_mutex;
double* g_vn_ptr[VN_MAX_DEVICES] = {};

int scratch_for_device(Model* m, double** out) {
  if (m->device < 0 || m->device >= VN_MAX_DEVICES) { m->err = "allegro_virial_noalloc: device ordinal out of range"; return ALLEGRO_ERR_UNSUPPORTED; }
  std::lock_guard<std::mutex> lock(g_vn_mutex);
  if (!g_vn_ptr[m->device]) {
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return cuda_fail(m, e, "allegro_virial_noalloc: cudaGetDevice");
    if (cur != m->device) { m->err = "allegro_virial_noalloc: the handle's device is not the current device"; return ALLEGRO_ERR_INVALID; }
    double* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_virial_scratch);
    if (e != cudaSuccess || !p) { cudaGetLastError(); return cuda_fail(m, e, "allegro_virial_noalloc: cudaGetSymbolAddress"); }
    g_vn_ptr[m->device] = p;
  }
  *out = g_vn_ptr[m->device];
  return 0;
}

}  // namespace

// Called from allegro_create (set-up, the handle's device current): the first allegro_virial_noalloc then does no symbol lookup.
int virial_noalloc_setup(Model* m) {
  double* p = nullptr;
  return scratch_for_device(m, &p);
}

}  // namespace allegro

extern "C" int allegro_virial_noalloc(void* h, const double* pos, double* W_out, void* stream) {
  using namespace allegro;
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!W_out) { m->err = "allegro_virial_noalloc: null output"; return ALLEGRO_ERR_INVALID; }
  if (!m->nl.valid) { m->err = "allegro_virial_noalloc called before a force evaluation"; return ALLEGRO_ERR_NO_LIST; }
  if (!pos && !m->md_ready) { m->err = "allegro_virial_noalloc: pos == NULL needs an MD state"; return ALLEGRO_ERR_INVALID; }
  const int64_t N = m->nl.N;
  if (N > VN_MAX_ATOMS) {
    m->err = "allegro_virial_noalloc: " + std::to_string(N) + " atoms exceed the fixed scratch array (ALLEGRO_VIRIAL_NOALLOC_MAX_ATOMS = " +
             std::to_string(VN_MAX_ATOMS) + "); use allegro_virial";
    return ALLEGRO_ERR_UNSUPPORTED;
  }
  double* scratch = nullptr;
  if (int rc = scratch_for_device(m, &scratch)) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const double* p = pos ? pos : m->md_pos.as<double>();
  const int nb = (int)((N + VN_ATOMS_PER_BLOCK - 1) / VN_ATOMS_PER_BLOCK);
  VnCell cl;
  for (int k = 0; k < 9; ++k) cl.H[k] = m->nl.H[k];
  if (nb > 0)
    k_virial_partial_na<<<nb, 256, 0, st>>>(m->nl.rowptr.as<int64_t>(), m->nl.keys.as<uint64_t>(), m->g_list.as<float>(), p, N, cl, scratch);
  k_virial_final_na<<<1, 288, 0, st>>>(scratch, nb, W_out);   // nb == 0 writes zeros
  m->launches += nb > 0 ? 2 : 1;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_virial_noalloc");
  return ALLEGRO_OK;
}
