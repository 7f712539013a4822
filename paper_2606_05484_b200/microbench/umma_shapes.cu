// microbenchmark: tcgen05.mma cta_group::2 throughput from shared memory for the RVQ score shape, with the descriptors
// REBUILT from addresses per MMA as the library's issue loops first did: N = 128 reads 75-108 cycles against a floor of 64
// because the one issuing thread spends that long between MMAs (umma_a_tmem.cu, with a clean loop, reaches 64); the RVQ
// scan loop now advances the descriptors' low words instead (umma_bf16_pair_lo in tc_common.cuh).
#include <cstdio>
#include "tc_common.cuh"
using namespace mapl::tc;
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(128, 1) k_mma(int N, int nkb, int chunks, int xstep, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;                       // nkb tiles [128 x 64] 16-bit
  uint8_t* sB = smem + 4 * 16384;           // nkb half tiles (N/2 rows)
  uint8_t* sX = sB + 4 * 16384;
  uint64_t* bar = reinterpret_cast<uint64_t*>(sX + 8192);
  uint32_t* slot = reinterpret_cast<uint32_t*>(bar + 4);
  const uint32_t rank = cluster_ctarank();
  for (int i = threadIdx.x; i < (4 * 16384 * 2 + 8192) / 4; i += 128) reinterpret_cast<uint32_t*>(smem)[i] = 0x3c003c00u;  // fp16 1.0
  if (threadIdx.x == 0) { mbar_init(&bar[0], 1); fence_barrier_init(); }
  fence_proxy_async_smem();
  if (threadIdx.x < 32) tmem_alloc_pair<512>(slot);
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem = *slot;
  if (rank == 0 && threadIdx.x == 32) {
    const uint32_t idesc = make_idesc_f16(256, N);
    long long t0 = clock64();
    for (int c = 0; c < chunks; ++c) {
      const uint32_t d = tmem + (c & 1) * 256;
      for (int kb = 0; kb < nkb; ++kb) {
        const uint32_t a = smem_u32(sA + kb * 16384), b = smem_u32(sB + kb * 16384);
#pragma unroll
        for (int k = 0; k < 4; ++k) umma_bf16_pair(d, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc, (kb | k) != 0);
      }
      if (xstep) umma_bf16_pair(d, desc_kmajor_sw32_k16(smem_u32(sX)), desc_kmajor_sw32_k16(smem_u32(sX + 4096)), idesc, 1);
    }
    long long t1 = clock64();
    umma_commit_pair(&bar[0]);
    mbar_wait(&bar[0], 0);
    long long t2 = clock64();
    out[0] = t1 - t0; out[1] = t2 - t0;
  }
  if (rank == 1 && threadIdx.x == 32) mbar_wait(&bar[0], 0);
  tc_fence_before_sync();
  cluster_sync_all();
  if (threadIdx.x < 32) { tc_fence_after_sync(); tmem_dealloc_pair<512>(tmem); }
}
int main() {
  long long* out; cudaMalloc(&out, 64);
  cudaFuncSetAttribute(k_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  for (int N : {128, 256}) for (int nkb : {1, 4}) for (int x : {0, 1}) {
    const int chunks = 200;
    for (int rep = 0; rep < 2; ++rep) k_mma<<<2, 128, 150 * 1024>>>(N, nkb, chunks, x, out);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("err %s\n", cudaGetErrorString(cudaGetLastError())); return 1; }
    long long h[2]; cudaMemcpy(h, out, 16, cudaMemcpyDeviceToHost);
    const int n_mma = chunks * (nkb * 4 + x);
    printf("N %3d nkb %d xstep %d: issue %6.1f cycles/MMA, complete %6.1f cycles/MMA (floor %d)\n", N, nkb, x, (double)h[0] / n_mma, (double)h[1] / n_mma, N / 2);
  }
  return 0;
}
