// microbenchmark: do tcgen05.mma (accumulating into TMEM) and tcgen05.ld (reading another TMEM region) share bandwidth?
#include <cstdio>
#include "tc_common.cuh"
using namespace mapl::tc;
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(320, 1) k_b(int N, int n_mma, int n_ld, long long* out, float* sink) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem; uint8_t* sB = smem + 6 * 16384;
  uint64_t* bar = reinterpret_cast<uint64_t*>(sB + 6 * 16384);
  uint32_t* slot = reinterpret_cast<uint32_t*>(bar + 4);
  const uint32_t rank = cluster_ctarank();
  const int warp = threadIdx.x / 32;
  for (int i = threadIdx.x; i < (12 * 16384) / 4; i += 320) reinterpret_cast<uint32_t*>(smem)[i] = 0x3c003c00u;
  if (threadIdx.x == 0) { mbar_init(&bar[0], 1); fence_barrier_init(); }
  fence_proxy_async_smem();
  if (warp == 1) tmem_alloc_pair<512>(slot);
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem = *slot;
  float acc = 0.f;
  long long t0 = clock64(), t_mma = 0, t_ld = 0;
  if (warp == 0 && threadIdx.x == 0 && rank == 0 && n_mma > 0) {
    const uint32_t idesc = make_idesc_f16(256, N);
    for (int i = 0; i < n_mma; ++i) {
      const int kb = i % 6;
      const uint32_t a = smem_u32(sA + kb * 16384), b = smem_u32(sB + kb * 16384);
#pragma unroll
      for (int k = 0; k < 4; ++k) umma_bf16_pair(tmem, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc, 1);
    }
    umma_commit_pair(&bar[0]);
    mbar_wait(&bar[0], 0);
    t_mma = clock64() - t0;
  }
  if (warp == 0 && threadIdx.x == 0 && rank == 1 && n_mma > 0) mbar_wait(&bar[0], 0);
  if (warp >= 2) {
    const uint32_t tr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + 256;
    for (int i = 0; i < n_ld; ++i) {
      uint32_t v[32], w[32];
      tmem_ld32(tr + (i & 3) * 64, v);
      tmem_ld32(tr + (i & 3) * 64 + 32, w);
      tmem_ld_wait();
      acc += __uint_as_float(v[0]) + __uint_as_float(w[31]);     // constant indices: v[i & 31] put both arrays in local memory
    }
    t_ld = clock64() - t0;
  }
  if (acc == 123.4f) sink[0] = acc;
  if (threadIdx.x == 0 && rank == 0) out[0] = t_mma;
  if (threadIdx.x == 64 && rank == 0) out[1] = t_ld;
  tc_fence_before_sync();
  cluster_sync_all();
  if (warp == 1) { tc_fence_after_sync(); tmem_dealloc_pair<512>(tmem); }
}
int main() {
  long long* out; cudaMalloc(&out, 64); float* sink; cudaMalloc(&sink, 64);
  cudaFuncSetAttribute(k_b, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
  const int n_mma = 400, n_ld = 400;   // 400 k-blocks of 4 MMAs; 400 x (2 x32 loads per warp) = 8 warps x 400 x 8 KB
  for (int N : {128, 256}) for (int mode : {1, 2, 3}) {
    cudaMemset(out, 0, 64);
    for (int rep = 0; rep < 2; ++rep) k_b<<<2, 320, 200 * 1024>>>(N, (mode & 1) ? n_mma : 0, (mode & 2) ? n_ld : 0, out, sink);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("err %s\n", cudaGetErrorString(cudaGetLastError())); return 1; }
    long long h[2]; cudaMemcpy(h, out, 16, cudaMemcpyDeviceToHost);
    printf("N %3d %s: MMA %7.1f cycles per k-block of 4 (floor %d) | LD %7.1f cycles per 64 KB read by the CTA (16 x32 loads)\n", N,
           mode == 1 ? "MMA alone " : mode == 2 ? "LD alone  " : "both      ", (double)h[0] / n_mma, N * 2, (double)h[1] / n_ld);
  }
  return 0;
}
