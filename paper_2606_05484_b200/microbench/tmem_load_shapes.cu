// microbenchmark: tcgen05.ld shapes: bytes per cycle per SM with 4 and 8 warps (one load + wait per iteration; `depth2`:
// two loads in flight before the wait).  The first version of this file consumed v[it & 31]: the run-time index put
// v[] in local memory, 32 STL per load went through the same LSU path, and every shape read "57 B/cycle" -- an artefact
// (profiles/r02_microbench.md keeps both outputs).
#include <cstdio>
#include "tc_common.cuh"
using namespace mapl::tc;
// each variant loads into 32 registers (128 B per thread = 4 KB per warp) unless noted
#define R32 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}"
#define O32 "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
template <int V>
__device__ __forceinline__ void ld(uint32_t a, uint32_t (&v)[32]) {
  if (V == 0) asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 " R32 ", [%32];" : O32 : "r"(a));
  if (V == 1) asm volatile("tcgen05.ld.sync.aligned.16x256b.x8.b32 " R32 ", [%32];" : O32 : "r"(a));     // 16 lanes x 64 cols
  if (V == 2) asm volatile("tcgen05.ld.sync.aligned.16x128b.x16.b32 " R32 ", [%32];" : O32 : "r"(a));    // 16 lanes x 64 cols
  if (V == 3) asm volatile("tcgen05.ld.sync.aligned.16x64b.x32.b32 " R32 ", [%32];" : O32 : "r"(a));     // 16 lanes x 64 cols
  if (V == 4) asm volatile("tcgen05.ld.sync.aligned.32x32b.pack::16b.x32.b32 " R32 ", [%32];" : O32 : "r"(a));   // 64 cols packed
}
template <int V>
__global__ void __launch_bounds__(512, 1) k_ld(int W, int iters, long long* out, float* sink) {
  __shared__ uint32_t slot;
  const int warp = threadIdx.x / 32;
  if (warp == 0) tmem_alloc<512>(&slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = slot + ((uint32_t)((warp & 3) * 32) << 16);
  float acc = 0.f;
  __syncthreads();
  long long t0 = clock64();
  if (warp < W) {
    for (int it = 0; it < iters; ++it) {
      uint32_t v[32];
      ld<V>(tmem + (it & 3) * 64, v);
      tmem_ld_wait();
      acc += __uint_as_float(v[0]) + __uint_as_float(v[31]);     // constant indices: a run-time index sends v[] to local memory
    }
  }
  __syncthreads();
  long long t1 = clock64();
  if (threadIdx.x == 0) out[0] = t1 - t0;
  if (acc == 123.456f) sink[0] = acc;
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(slot);
}
__global__ void __launch_bounds__(512, 1) k_ld2(int W, int iters, long long* out, float* sink) {
  __shared__ uint32_t slot;
  const int warp = threadIdx.x / 32;
  if (warp == 0) tmem_alloc<512>(&slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = slot + ((uint32_t)((warp & 3) * 32) << 16);
  float acc = 0.f;
  __syncthreads();
  long long t0 = clock64();
  if (warp < W) {
    for (int it = 0; it < iters; ++it) {
      uint32_t v[32], w[32];
      ld<0>(tmem + (it & 3) * 64, v);
      ld<0>(tmem + (it & 3) * 64 + 32, w);
      tmem_ld_wait();
      acc += __uint_as_float(v[0]) + __uint_as_float(w[31]);
    }
  }
  __syncthreads();
  long long t1 = clock64();
  if (threadIdx.x == 0) out[0] = t1 - t0;
  if (acc == 123.456f) sink[0] = acc;
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(slot);
}
template <int V>
void run(const char* name, double cells_per_load, long long* out, float* sink) {
  for (int W : {4, 8}) {
    const int iters = 1000;
    for (int rep = 0; rep < 2; ++rep) k_ld<V><<<1, 512>>>(W, iters, out, sink);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("%s err %s\n", name, cudaGetErrorString(cudaGetLastError())); return; }
    long long h; cudaMemcpy(&h, out, 8, cudaMemcpyDeviceToHost);
    printf("%-26s W %d: %7.1f cycles per load per warp, %6.1f TMEM cells (4 B) per cycle per SM\n", name, W, (double)h / iters, W * iters * cells_per_load / h);
  }
}
int main() {
  long long* out; cudaMalloc(&out, 64); float* sink; cudaMalloc(&sink, 64);
  run<0>("32x32b.x32 (32 lanes x 32c)", 1024, out, sink);
  run<1>("16x256b.x8 (16 lanes x 64c)", 1024, out, sink);
  run<2>("16x128b.x16", 1024, out, sink);
  run<3>("16x64b.x32", 1024, out, sink);
  run<4>("32x32b.pack16.x32 (64c)", 2048, out, sink);
  for (int W : {4, 8}) {
    const int iters = 1000;
    for (int rep = 0; rep < 2; ++rep) k_ld2<<<1, 512>>>(W, iters, out, sink);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("depth2 err %s\n", cudaGetErrorString(cudaGetLastError())); return 1; }
    long long h; cudaMemcpy(&h, out, 8, cudaMemcpyDeviceToHost);
    printf("%-26s W %d: %7.1f cycles per pair of loads per warp, %6.1f TMEM cells (4 B) per cycle per SM\n", "32x32b.x32 depth2", W, (double)h / iters, W * iters * 2048.0 / h);
  }
  return 0;
}
