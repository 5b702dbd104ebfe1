// tp3_fwd.cu — instantiations of the few-channel forward tensor-product kernel (tp3.cuh), one per layer signature of
// tp_gen.cuh; lmax <= 2 signatures also get the channel count (8, 16, 32) as a compile-time constant.  A translation
// unit of its own so that the two directions compile in parallel.
#include "tp3.cuh"

namespace allegro {

template <int SIG, int NCH>
static void launch_t(int grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io) {
  static int attr_dev = -1;   // the attribute is per device
  int dev = 0;
  cudaGetDevice(&dev);
  if (attr_dev != dev) { cudaFuncSetAttribute(k_tp_fwd3<SIG, NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); attr_dev = dev; }
  k_tp_fwd3<SIG, NCH><<<grid, 256, smem, st>>>(tp, io);
}
template <int SIG>
static void launch_sig(int grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io) {
  if constexpr (tpgen::SigDims<SIG>::LMAX <= 2) {
    switch (tp.n) {
      case 8: launch_t<SIG, 8>(grid, smem, st, tp, io); return;
      case 16: launch_t<SIG, 16>(grid, smem, st, tp, io); return;
      case 32: launch_t<SIG, 32>(grid, smem, st, tp, io); return;
      default: break;
    }
  }
  launch_t<SIG, 0>(grid, smem, st, tp, io);
}

void launch_tp3_fwd(int sig, int grid, size_t smem, cudaStream_t st, const TpLayerDev& tp, const TpIo& io) {
  switch (sig) {
#define X(I) case I: launch_sig<I>(grid, smem, st, tp, io); break;
    TPGEN_FOR_EACH_SIG(X)
#undef X
    default: break;
  }
}

}  // namespace allegro
