// microbenchmark 3: per-instruction cost seen by a single producer thread
#include <cstdio>
#include <vector>
#include "tc_common.cuh"
using namespace mapl::tc;

__global__ void __launch_bounds__(64, 1) k_bench(const __grid_constant__ CUtensorMap tm, int rows_total, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + (size_t)16 * 8192);
  if (threadIdx.x == 0) {
    for (int i = 0; i < 64; ++i) mbar_init(&bar[i], 1);
    fence_barrier_init();
  }
  __syncthreads();
  if (threadIdx.x != 0) return;
  const int N = 64;
  long long t[8];
  // a) waits on a barrier whose phase 1 counts as complete
  t[0] = clock64();
  for (int i = 0; i < N; ++i) mbar_wait(&bar[0], 1);
  t[1] = clock64();
  // b) arrive.expect_tx(0) alone
  for (int i = 0; i < N; ++i) mbar_arrive_expect_tx(&bar[1], 0);
  t[2] = clock64();
  // c) N TMA loads back to back on one barrier
  mbar_arrive_expect_tx(&bar[2], 8192 * N);
  for (int i = 0; i < N; ++i) tma_load_2d(smem + (size_t)(i % 16) * 8192, &tm, &bar[2], 0, (i * 64) % (rows_total - 64), kEvictLast);
  t[3] = clock64();
  mbar_wait(&bar[2], 0);
  t[4] = clock64();
  // d) expect_tx + TMA per iteration, a barrier each (no waits)
  for (int i = 0; i < 32; ++i) {
    mbar_arrive_expect_tx(&bar[3 + i], 8192);
    tma_load_2d(smem + (size_t)(i % 16) * 8192, &tm, &bar[3 + i], 0, (i * 64) % (rows_total - 64), kEvictLast);
  }
  t[5] = clock64();
  for (int i = 0; i < 32; ++i) mbar_wait(&bar[3 + i], 0);
  t[6] = clock64();
  out[0] = (t[1] - t[0]) / N; out[1] = (t[2] - t[1]) / N; out[2] = (t[3] - t[2]) / N; out[3] = t[4] - t[3];
  out[4] = (t[5] - t[4]) / 32; out[5] = t[6] - t[5];
}

int main() {
  const int rows_total = 8192;
  void* buf; cudaMalloc(&buf, (size_t)rows_total * 128); cudaMemset(buf, 1, (size_t)rows_total * 128);
  long long* out; cudaMalloc(&out, 64 * 8);
  cudaFuncSetAttribute(k_bench, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  CUtensorMap tm;
  if (!make_tmap_bf16_2d(&tm, buf, rows_total, 64, 64, 64, 64)) return 1;
  size_t smem = (size_t)16 * 8192 + 1024 + 1024;
  for (int rep = 0; rep < 3; ++rep) {
    k_bench<<<1, 64, smem>>>(tm, rows_total, out);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { printf("err %s\n", cudaGetErrorString(e)); return 1; }
    long long h[8]; cudaMemcpy(h, out, 64, cudaMemcpyDeviceToHost);
    printf("wait(done) %lld | expect_tx %lld | TMA issue b2b %lld (+ drain %lld) | expect+TMA %lld (+ drain %lld)\n", h[0], h[1], h[2], h[3], h[4], h[5]);
  }
  return 0;
}
