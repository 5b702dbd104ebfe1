// L2 -> SM bandwidth probe: every CTA streams the same small (L2-resident) buffer through a shared-memory ring with cp.async.bulk
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  }
}
template <int CL>
__global__ void k_bulk(const uint8_t* __restrict__ buf, size_t bufbytes, int chunk, int ring, int iters, unsigned long long* sink) {
  extern __shared__ __align__(1024) uint8_t sm[];
  __shared__ __align__(8) uint64_t bar[16];
  uint32_t rank = 0;
  if (CL > 1) asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
  if (threadIdx.x == 0) { for (int i = 0; i < ring; ++i) mbar_init(&bar[i], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  __syncthreads();
  if (CL > 1) { asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory"); }
  const int nchunks = (int)(bufbytes / chunk);
  if (CL == 1) {
    if (threadIdx.x == 0) {
      int issued = 0, waited = 0;
      const int total = iters * nchunks;
      int c0 = (blockIdx.x * 7) % nchunks;
      while (waited < total) {
        while (issued < total && issued - waited < ring) {
          const int slot = issued % ring;
          const uint8_t* src = buf + (size_t)((c0 + issued) % nchunks) * chunk;
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar[slot])), "r"(chunk) : "memory");
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(sm + (size_t)slot * chunk)), "l"(src), "r"(chunk), "r"(smem_u32(&bar[slot])) : "memory");
          ++issued;
        }
        mbar_wait(&bar[waited % ring], (uint32_t)((waited / ring) & 1));
        ++waited;
      }
      sink[blockIdx.x] = sm[0];
    }
  } else {
    // lock-step rounds of `ring` chunks: every CTA loads 1/CL of each chunk and multicasts it to the whole cluster
    const int total = iters * nchunks;
    int c0 = (blockIdx.x / CL * 7) % nchunks;
    const int part = chunk / CL;
    int round = 0;
    for (int base = 0; base < total; base += ring, ++round) {
      const int cnt = min(ring, total - base);
      if (threadIdx.x == 0) {
        for (int s2 = 0; s2 < cnt; ++s2) {
          const uint8_t* src = buf + (size_t)((c0 + base + s2) % nchunks) * chunk;
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&bar[s2])), "r"(chunk) : "memory");
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1], %2, [%3], %4;" ::"r"(smem_u32(sm + (size_t)s2 * chunk + rank * part)), "l"(src + rank * part), "r"(part), "r"(smem_u32(&bar[s2])), "h"((uint16_t)((1 << CL) - 1)) : "memory");
        }
        for (int s2 = 0; s2 < cnt; ++s2) mbar_wait(&bar[s2], (uint32_t)(round & 1));
      }
      __syncthreads();
      asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    if (threadIdx.x == 0) sink[blockIdx.x] = sm[0];
  }
}
__global__ void k_ldg(const uint4* __restrict__ buf, size_t n16, int iters, unsigned long long* sink) {
  uint4 acc = make_uint4(0, 0, 0, 0);
  const size_t stride = blockDim.x;
  for (int it = 0; it < iters; ++it) {
    size_t i = threadIdx.x + ((size_t)blockIdx.x * 9973 * 64) % n16;
    for (size_t k = 0; k < n16; k += stride * 4) {
      uint4 a = buf[(i + k) % n16], b = buf[(i + k + stride) % n16], c = buf[(i + k + 2 * stride) % n16], d = buf[(i + k + 3 * stride) % n16];
      acc.x ^= a.x ^ b.x ^ c.x ^ d.x; acc.y ^= a.y ^ b.y ^ c.y ^ d.y;
    }
  }
  if (acc.x == 0x12345678 && acc.y == 77) sink[0] = acc.x;
}
int main() {
  int dev = 0; cudaSetDevice(dev);
  cudaDeviceProp p; cudaGetDeviceProperties(&p, dev);
  int clk = 0; cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, dev);
  printf("%s SMs=%d clock %d kHz\n", p.name, p.multiProcessorCount, clk);
  const size_t bufbytes = 3 << 20;
  uint8_t* buf; cudaMalloc(&buf, bufbytes); cudaMemset(buf, 1, bufbytes);
  unsigned long long* sink; cudaMalloc(&sink, 8 * 4096);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  auto run = [&](int CL, int per_sm, int chunk, int ring, int iters) {
    const int grid = p.multiProcessorCount * per_sm;
    const size_t smem = (size_t)chunk * ring;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
      cudaEventRecord(e0);
      if (CL == 1) { cudaFuncSetAttribute(k_bulk<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); k_bulk<1><<<grid, 64, smem>>>(buf, bufbytes, chunk, ring, iters, sink); }
      else {
        cudaLaunchConfig_t cfg{}; cfg.gridDim = dim3(grid); cfg.blockDim = dim3(64); cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute at[1]; at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        if (CL == 2) { cudaFuncSetAttribute(k_bulk<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); cudaLaunchKernelEx(&cfg, k_bulk<2>, (const uint8_t*)buf, bufbytes, chunk, ring, iters, sink); }
        else { cudaFuncSetAttribute(k_bulk<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); cudaLaunchKernelEx(&cfg, k_bulk<4>, (const uint8_t*)buf, bufbytes, chunk, ring, iters, sink); }
      }
      cudaEventRecord(e1); cudaEventSynchronize(e1);
      float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    cudaError_t e = cudaGetLastError();
    const double bytes = (double)grid * iters * bufbytes;   // bytes delivered to shared memory
    printf("bulk CL=%d ctas/sm=%d chunk=%5d ring=%d : %.3f ms  delivered %.2f TB/s  (%.1f B/clk/SM @1.9GHz) l2-requested %.2f TB/s %s\n", CL, per_sm, chunk, ring, best,
           bytes / best / 1e9, bytes / best / 1e9 * 1e12 / 148 / 1.9e9, bytes / CL / best / 1e9, e == cudaSuccess ? "" : cudaGetErrorString(e));
  };
  for (int per_sm : {1, 2})
    for (int chunk : {8192, 16384, 32768})
      for (int ring : {2, 4, 6}) {
        if ((size_t)chunk * ring * per_sm > 200 * 1024) continue;
        run(1, per_sm, chunk, ring, 20);
      }
  for (int CL : {2, 4})
    for (int chunk : {16384, 32768})
      for (int ring : {3, 6}) run(CL, 1, chunk, ring, 20);
  for (int threads : {256, 1024}) {
    const int grid = p.multiProcessorCount * (2048 / threads);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
      cudaEventRecord(e0);
      k_ldg<<<grid, threads>>>((const uint4*)buf, bufbytes / 16, 10, sink);
      cudaEventRecord(e1); cudaEventSynchronize(e1);
      float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    printf("ldg.128 threads=%d grid=%d: %.3f ms %.2f TB/s\n", threads, grid, best, (double)grid * 10 * bufbytes / best / 1e9);
  }
  return 0;
}
