// probe 3: tcgen05.mma issue rate (cycles per MMA) for tf32 / f16, A from shared memory or TMEM, with and without concurrent bulk copies
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ bool mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  for (int it = 0; it < 2000000 && !done; ++it)
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return done != 0;
}
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}
template <int KIND>
__device__ __forceinline__ void mma_ss(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
  if (KIND == 0) asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"(acc));
  else asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"(acc));
}
template <int KIND>
__device__ __forceinline__ void mma_ts(uint32_t d, uint32_t a_tmem, uint64_t b, uint32_t idesc, uint32_t acc) {
  if (KIND == 0) asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d), "r"(a_tmem), "l"(b), "r"(idesc), "r"(acc));
  else asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d), "r"(a_tmem), "l"(b), "r"(idesc), "r"(acc));
}
// one K step = 32 bytes of K per row (8 tf32 / 16 f16).  B tile: N rows x 32 B, A tile: 128 rows x 32 B, canonical no-swizzle K-major.
template <int KIND, int ATMEM>
__global__ void __launch_bounds__(192) k_mma(int N, int nmma_per_commit, int ncommits, int load_chunk, unsigned long long* out) {
  extern __shared__ __align__(1024) uint8_t sm[];
  __shared__ __align__(8) uint64_t bar_mma[2];
  __shared__ __align__(8) uint64_t bar_ld[16];
  __shared__ uint32_t tmem_base_s;
  __shared__ volatile int stop_flag;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (threadIdx.x == 0) {
    mbar_init(&bar_mma[0], 1); mbar_init(&bar_mma[1], 1);
    for (int i = 0; i < 16; ++i) mbar_init(&bar_ld[i], 1);
    stop_flag = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // zero the operand area (A 2 x 4 KB, B 2 x N x 32 B)
  for (int i = threadIdx.x; i < (2 * 4096 + 2 * N * 32) / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(sm)[i] = 0x3c003c00u;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_base_s;
  uint8_t* ldbuf = sm + 2 * 4096 + 2 * N * 32;
  if (warp == 0) {
    if (lane == 0) {
      const uint32_t idesc = (1u << 4) | ((KIND == 0 ? 2u : 0u) << 7) | ((KIND == 0 ? 2u : 0u) << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
      const uint32_t sa = smem_u32(sm), sb = smem_u32(sm + 2 * 4096);
      const uint64_t dA0 = umma_desc(sa, 128, 256), dA1 = umma_desc(sa + 4096, 128, 256);
      const uint64_t dB0 = umma_desc(sb, 128, 256), dB1 = umma_desc(sb + N * 32, 128, 256);
      const uint32_t aT0 = tmem + 256, aT1 = tmem + 256 + 8;    // A operand columns (accumulator at columns [0, N))
      bool ok = true;
      const long long t0 = clock64();
      for (int c = 0; c < ncommits && ok; ++c) {
        if (c >= 2) ok = mbar_wait(&bar_mma[c & 1], (uint32_t)(((c >> 1) - 1) & 1));
        for (int i = 0; i < nmma_per_commit; i += 3) {
          if (ATMEM) {
            mma_ts<KIND>(tmem, aT1, dB0, idesc, 1u);
            mma_ts<KIND>(tmem, aT0, dB1, idesc, 1u);
            mma_ts<KIND>(tmem, aT0, dB0, idesc, 1u);
          } else {
            mma_ss<KIND>(tmem, dA1, dB0, idesc, 1u);
            mma_ss<KIND>(tmem, dA0, dB1, idesc, 1u);
            mma_ss<KIND>(tmem, dA0, dB0, idesc, 1u);
          }
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar_mma[c & 1])) : "memory");
      }
      for (int c = ncommits - 2; c < ncommits && ok; ++c) if (c >= 0) ok = mbar_wait(&bar_mma[c & 1], (uint32_t)((c >> 1) & 1));
      const long long t1 = clock64();
      stop_flag = 1;
      out[blockIdx.x * 4 + 0] = ok ? (unsigned long long)(t1 - t0) : 0ull;
    }
  } else if (warp >= 2 && load_chunk > 0) {
    // four loader warps, each with a private 2-slot ring, run until the MMA thread is done
    if (lane == 0) {
      const int w = warp - 2;
      uint8_t* base = ldbuf + (size_t)w * 2 * load_chunk;
      uint64_t* b = bar_ld + w * 2;
      const uint8_t* src = reinterpret_cast<const uint8_t*>(out) + 65536;   // any readable memory: the buffer behind `out`
      unsigned long long n = 0;
      int issued = 0, waited = 0;
      bool ok = true;
      while (ok && (!stop_flag || waited < issued)) {
        while (!stop_flag && issued - waited < 2) {
          const int slot = issued & 1;
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&b[slot])), "r"(load_chunk) : "memory");
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(base + (size_t)slot * load_chunk)), "l"(src + (size_t)((issued * 4 + w) % 32) * load_chunk), "r"(load_chunk), "r"(smem_u32(&b[slot])) : "memory");
          ++issued;
        }
        if (waited < issued) { ok = mbar_wait(&b[waited & 1], (uint32_t)((waited >> 1) & 1)); ++waited; ++n; }
      }
      out[blockIdx.x * 4 + 1 + (w & 1)] = n;   // two of the four counters are enough
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
}
template <int KIND, int ATMEM>
void run(const char* name, int N, int load_chunk, unsigned long long* d_out, unsigned long long* h_out) {
  const int nmma = 96, ncommits = 400;
  const size_t smem = 2 * 4096 + 2 * (size_t)N * 32 + 8 * (size_t)load_chunk + 1024;
  cudaFuncSetAttribute(k_mma<KIND, ATMEM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  cudaMemset(d_out, 0, 148 * 4 * 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0);
  k_mma<KIND, ATMEM><<<148, 192, smem>>>(N, nmma, ncommits, load_chunk, d_out);
  cudaEventRecord(e1);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
  cudaMemcpy(h_out, d_out, 148 * 4 * 8, cudaMemcpyDeviceToHost);
  double cyc = 0, ld = 0; int bad = 0;
  for (int b = 0; b < 148; ++b) { cyc += (double)h_out[b * 4]; ld += (double)(h_out[b * 4 + 1] + h_out[b * 4 + 2]) * 2; if (!h_out[b * 4]) ++bad; }
  cyc /= 148; ld /= 148;
  const double per_mma = cyc / ((double)nmma * ncommits);
  const double flops = 148.0 * nmma * ncommits * 2.0 * 128 * N * (KIND == 0 ? 8 : 16);
  printf("%-14s N=%3d load_chunk=%5d: %.3f ms  %.1f cyc/MMA (ideal %d)  %.0f TFLOP/s dense  loads %.1f B/clk/SM  bad=%d %s\n", name, N, load_chunk, ms, per_mma, N / 2,
         flops / ms / 1e9, ld * load_chunk / (cyc > 0 ? cyc : 1), bad, cudaGetErrorString(e));
}
int main() {
  cudaSetDevice(0);
  unsigned long long* d_out; cudaMalloc(&d_out, 4 << 20); cudaMemset(d_out, 0, 4 << 20);
  unsigned long long h_out[148 * 4];
  for (int chunk : {0, 8192, 16384}) {
    for (int N : {256, 192, 128, 64}) {
      run<0, 0>("tf32 SS", N, chunk, d_out, h_out);
      run<0, 1>("tf32 TS(A tmem)", N, chunk, d_out, h_out);
      run<1, 0>("f16 SS", N, chunk, d_out, h_out);
      run<1, 1>("f16 TS(A tmem)", N, chunk, d_out, h_out);
    }
  }
  return 0;
}
