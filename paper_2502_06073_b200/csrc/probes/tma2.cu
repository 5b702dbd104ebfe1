// probe 2: (a) bulk copies issued by several warps of one CTA, (b) large chunks, (c) 2D TMA tensor loads with SWIZZLE_128B
#include <cstdio>
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
}
// nw issuing warps, each with its own ring of `ring` slots of `chunk` bytes
__global__ void k_bulk(const uint8_t* __restrict__ buf, size_t bufbytes, int chunk, int ring, int iters, unsigned long long* sink) {
  extern __shared__ __align__(1024) uint8_t sm[];
  __shared__ __align__(8) uint64_t bar[64];
  const int warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (threadIdx.x == 0) { for (int i = 0; i < nw * ring; ++i) mbar_init(&bar[i], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  __syncthreads();
  const int nchunks = (int)(bufbytes / chunk);
  if ((threadIdx.x & 31) == 0) {
    uint8_t* base = sm + (size_t)warp * ring * chunk;
    uint64_t* b = bar + warp * ring;
    int issued = 0, waited = 0;
    const int total = iters * nchunks / nw;
    int c0 = (blockIdx.x * 7 + warp * 13) % nchunks;
    while (waited < total) {
      while (issued < total && issued - waited < ring) {
        const int slot = issued % ring;
        const uint8_t* src = buf + (size_t)((c0 + issued) % nchunks) * chunk;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&b[slot])), "r"(chunk) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(base + (size_t)slot * chunk)), "l"(src), "r"(chunk), "r"(smem_u32(&b[slot])) : "memory");
        ++issued;
      }
      mbar_wait(&b[waited % ring], (uint32_t)((waited / ring) & 1));
      ++waited;
    }
    sink[blockIdx.x] = base[0];
  }
}
// 2D tensor loads: box = 32 floats x rows, SWIZZLE_128B; one issuing thread, ring slots
__global__ void k_tma(const __grid_constant__ CUtensorMap tm, int rows_total, int box_rows, int kcols, int ring, int iters, unsigned long long* sink) {
  extern __shared__ __align__(1024) uint8_t sm[];
  __shared__ __align__(8) uint64_t bar[16];
  if (threadIdx.x == 0) { for (int i = 0; i < ring; ++i) mbar_init(&bar[i], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  __syncthreads();
  const int bytes = box_rows * 128;
  if (threadIdx.x == 0) {
    const int ntiles = rows_total / box_rows, nk = kcols / 32;
    int issued = 0, waited = 0;
    const int total = iters;
    int t0 = blockIdx.x;
    while (waited < total) {
      while (issued < total && issued - waited < ring) {
        const int slot = issued % ring;
        const int idx = t0 * nk + issued;   // walk k blocks of this CTA's row tile, then the next tile
        const int tile = (idx / nk) % ntiles, kb = idx % nk;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar[slot])), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(sm + (size_t)slot * bytes)), "l"(&tm), "r"(kb * 32), "r"(tile * box_rows), "r"(smem_u32(&bar[slot])) : "memory");
        ++issued;
      }
      mbar_wait(&bar[waited % ring], (uint32_t)((waited / ring) & 1));
      ++waited;
    }
    sink[blockIdx.x] = sm[0];
  }
}
typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int main() {
  cudaSetDevice(0);
  cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
  const size_t bufbytes = 3 << 20;
  uint8_t* buf; cudaMalloc(&buf, bufbytes); cudaMemset(buf, 1, bufbytes);
  unsigned long long* sink; cudaMalloc(&sink, 8 * 4096);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaFuncSetAttribute(k_bulk, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
  cudaFuncSetAttribute(k_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
  for (int nw : {1, 2, 4})
    for (int chunk : {4096, 16384, 32768, 65536}) {
      for (int ring : {1, 2, 3}) {
        const size_t smem = (size_t)chunk * ring * nw;
        if (smem > 200 * 1024) continue;
        const int iters = 24, grid = p.multiProcessorCount;
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {
          cudaEventRecord(e0);
          k_bulk<<<grid, 32 * nw, smem>>>(buf, bufbytes, chunk, ring, iters, sink);
          cudaEventRecord(e1); cudaEventSynchronize(e1);
          float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
        }
        const double bytes = (double)grid * (iters * (bufbytes / chunk) / nw) * nw * chunk;
        const double per_op_ns = best * 1e6 / (iters * (bufbytes / chunk) / nw);
        printf("bulk warps=%d chunk=%6d ring=%d: %.3f ms %.2f TB/s  %.1f B/clk/SM  per-op(per warp) %.0f ns %s\n", nw, chunk, ring, best, bytes / best / 1e9,
               bytes / best / 1e9 * 1e12 / 148 / 1.9e9, per_op_ns, cudaGetErrorString(cudaGetLastError()));
      }
    }
  // ---- 2D tensor maps over a big fp32 matrix [rows][kcols]
  EncodeFn enc = nullptr; cudaDriverEntryPointQueryResult qres;
  cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &qres);
  if (!enc) { printf("no cuTensorMapEncodeTiled\n"); return 0; }
  const int rows = 1 << 18, kcols = 512;
  float* A; cudaMalloc(&A, (size_t)rows * kcols * 4); cudaMemset(A, 0, (size_t)rows * kcols * 4);
  for (int box_rows : {64, 128, 256}) {
    CUtensorMap tm;
    cuuint64_t gdim[2] = {(cuuint64_t)kcols, (cuuint64_t)rows};
    cuuint64_t gstr[1] = {(cuuint64_t)kcols * 4};
    cuuint32_t box[2] = {32, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, A, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { printf("encode failed %d\n", (int)r); continue; }
    for (int ring : {1, 2, 4, 8}) {
      const int bytes = box_rows * 128;
      if ((size_t)bytes * ring > 200 * 1024) continue;
      const int iters = 2048, grid = p.multiProcessorCount;
      float best = 1e30f;
      for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        k_tma<<<grid, 32, (size_t)bytes * ring>>>(tm, rows, box_rows, kcols, ring, iters, sink);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
      }
      const double tot = (double)grid * iters * bytes;
      printf("tma2d box=32x%3d ring=%d: %.3f ms %.2f TB/s %.1f B/clk/SM per-op %.0f ns %s\n", box_rows, ring, best, tot / best / 1e9, tot / best / 1e9 * 1e12 / 148 / 1.9e9,
             best * 1e6 / iters, cudaGetErrorString(cudaGetLastError()));
    }
  }
  return 0;
}
