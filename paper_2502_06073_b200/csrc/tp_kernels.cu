// tp_kernels.cu — instantiations of the generated tensor-product kernels (tp.cuh, tp3.cuh) and their launchers, in a
// translation unit of their own: one instantiation per layer signature of tp_gen.cuh.
#include <algorithm>

#include "tp_big.cuh"

namespace allegro {

// launch the generated instantiation of the tensor-product kernels for layer signature `sig`
void launch_tp_fwd(int sig, dim3 grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, int TE, int PC) {
  static int attr[tpgen::N_SIGS] = {0};   // device ordinal + 1 the attribute was last set on (it is per device)
  int dev = 0;
  cudaGetDevice(&dev);
  switch (sig) {
#define X(I)                                                                                                        \
  case I:                                                                                                           \
    if (attr[I] != dev + 1) { cudaFuncSetAttribute(k_tp_fwd<I>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); attr[I] = dev + 1; } \
    k_tp_fwd<I><<<grid, TP_T, smem, st>>>(tp, io, TE, PC);                                                            \
    break;
    TPGEN_FOR_EACH_SIG(X)
#undef X
    default: break;
  }
}
void launch_tp_bwd(int sig, dim3 grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, int TE, int d3max, int PC) {
  static int attr[tpgen::N_SIGS] = {0};   // device ordinal + 1 the attribute was last set on (it is per device)
  int dev = 0;
  cudaGetDevice(&dev);
  switch (sig) {
#define X(I)                                                                                                        \
  case I:                                                                                                           \
    if (attr[I] != dev + 1) { cudaFuncSetAttribute(k_tp_bwd<I>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024); attr[I] = dev + 1; } \
    k_tp_bwd<I><<<grid, TP_T, smem, st>>>(tp, io, TE, d3max, PC);                                                     \
    break;
    TPGEN_FOR_EACH_SIG(X)
#undef X
    default: break;
  }
}


// shared-memory bytes of the few-channel kernels (tp3.cuh); 0 when the layer has no channel mixing
size_t tp3_smem_bytes(const TpLayerDev& tp, bool backward) {
  if (!tp.has_lin) return 0;
  const int n = tp.n, TE = 256 / n;
  size_t f = 0;
  for (int o = 0; o < tp.n_out; ++o) {
    if (tp.out_off[o] < 0) continue;
    const size_t K = (size_t)tp.out_np[o] * n, rows = tp3_round16(TE * tp.out_d3[o]);
    f += backward ? 2 * n * (K + 8) + rows * (n + 4) + rows * (K + 4) : 2 * K * (n + 8) + rows * (K + 4);
  }
  return f * sizeof(float);
}

bool tp3_supported(const TpLayerDev& tp) {
  const int n = tp.n;
  if (!(n == 8 || n == 16 || n == 32) || tp.n_out > TP3_MAXO) return false;
  return tp3_smem_bytes(tp, true) <= 200 * 1024 && tp3_smem_bytes(tp, false) <= 200 * 1024;
}

void launch_tp3_fwd(int sig, int grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io);   // tp3_fwd.cu
void launch_tp3_bwd(int sig, int grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io);   // tp3_bwd.cu

void launch_tp3(int sig, bool backward, int grid, cudaStream_t st, const TpLayerDev& tp, const TpIo& io) {
  const size_t smem = tp3_smem_bytes(tp, backward);
  if (backward) launch_tp3_bwd(sig, grid, smem, st, tp, io);
  else launch_tp3_fwd(sig, grid, smem, st, tp, io);
}

// ---- many-channel path (tp_big.cuh)
bool tpbig_supported(const TpLayerDev& tp) { return (tp.n == 64 || tp.n == 128 || tp.n == 256) && tp.n_out <= TP3_MAXO; }

size_t tpbig_floats_per_edge(const TpLayerDev& tp) {
  if (!tp.has_lin) return 0;
  size_t f = 0;
  for (int o = 0; o < tp.n_out; ++o)
    if (tp.out_off[o] >= 0) f += (size_t)tp.out_d3[o] * tp.out_np[o] * tp.n;
  return f;
}

// backward: the ring kernel (T-bar staged by bulk copies) when at least two slots fit into shared memory, else k_tpo_bwd
template <int SIG>
bool launch_tpo_bwd_ring(cudaStream_t st, const TpLayerDev& tp, const TpIo& io, const TpBig& big) {
  static int sms[64] = {0};
  static bool attr[64] = {false};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return false;
  if (!tp.has_lin || tp.n > 256 || 256 % tp.n) return false;
  const size_t slot = TpoRing<SIG>::SLOT;
  int n_slots = (int)std::min<size_t>(TPO_RING_MAX_SLOTS, (220 * 1024 - 128) / slot);
  if (n_slots < 2) return false;
  const size_t smem = (size_t)n_slots * slot + 128;
  if (!attr[dev]) {
    if (cudaFuncSetAttribute(k_tpo_bwd_ring<SIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024) != cudaSuccess) { cudaGetLastError(); return false; }
    cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev);
    attr[dev] = true;
  }
  k_tpo_bwd_ring<SIG><<<(unsigned)std::max(1, sms[dev]), TPO_RING_T, smem, st>>>(tp, io, big, n_slots);
  return true;
}

void launch_tpo(int sig, bool backward, int64_t m_cap, cudaStream_t st, const TpLayerDev& tp, const TpIo& io, const TpBig& big) {
  const unsigned grid = (unsigned)((m_cap * tp.n + 255) / 256);
  switch (sig) {
#define X(I)                                                                                         \
  case I:                                                                                            \
    if (!backward) k_tpo_fwd<I><<<grid, 256, 0, st>>>(tp, io, big);                                 \
    else if (!launch_tpo_bwd_ring<I>(st, tp, io, big)) k_tpo_bwd<I><<<grid, 256, 0, st>>>(tp, io, big); \
    break;
    TPGEN_FOR_EACH_SIG(X)
#undef X
    default: break;
  }
}

}  // namespace allegro
