// microbenchmark 4: steady-state ring with waits: try_wait vs test_wait polling, depth 8
#include <cstdio>
#include "tc_common.cuh"
using namespace mapl::tc;
__device__ __forceinline__ void mbar_poll(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done)
    asm volatile("{\n.reg .pred p;\nmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.b32 %0, 1, 0, p;\n}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__global__ void __launch_bounds__(64, 1) k_bench(const __grid_constant__ CUtensorMap tm, int rows_total, int depth, int poll, long long* out, long long* lat) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + (size_t)16 * 8192);
  if (threadIdx.x == 0) { for (int i = 0; i < 64; ++i) mbar_init(&bar[i], 1); fence_barrier_init(); }
  __syncthreads();
  if (threadIdx.x != 0) return;
  const int N = 128;
  long long t0 = clock64(), waited = 0;
  for (int it = 0; it < N + depth; ++it) {
    const int s = it % depth;
    if (it >= depth) {
      long long a = clock64();
      if (poll) mbar_poll(&bar[s], ((it - depth) / depth) & 1); else mbar_wait(&bar[s], ((it - depth) / depth) & 1);
      waited += clock64() - a;
    }
    if (it < N) {
      mbar_arrive_expect_tx(&bar[s], 8192);
      tma_load_2d(smem + (size_t)s * 8192, &tm, &bar[s], 0, (it * 64) % (rows_total - 64), kEvictLast);
    }
  }
  out[0] = (clock64() - t0) / N; out[1] = waited / N;
}
int main() {
  const int rows_total = 8192;
  void* buf; cudaMalloc(&buf, (size_t)rows_total * 128); cudaMemset(buf, 1, (size_t)rows_total * 128);
  long long* out; cudaMalloc(&out, 64 * 8);
  cudaFuncSetAttribute(k_bench, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  CUtensorMap tm;
  if (!make_tmap_bf16_2d(&tm, buf, rows_total, 64, 64, 64, 64)) return 1;
  size_t smem = (size_t)16 * 8192 + 1024 + 1024;
  for (int depth : {1, 2, 4, 8, 16}) for (int poll : {0, 1}) {
    for (int rep = 0; rep < 2; ++rep) k_bench<<<1, 64, smem>>>(tm, rows_total, depth, poll, out, out + 8);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("err\n"); return 1; }
    long long h[2]; cudaMemcpy(h, out, 16, cudaMemcpyDeviceToHost);
    printf("depth %2d %s: %lld cycles/op, of which waiting %lld\n", depth, poll ? "test_wait poll" : "try_wait     ", h[0], h[1]);
  }
  return 0;
}
