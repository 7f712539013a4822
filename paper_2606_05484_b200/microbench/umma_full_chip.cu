// microbenchmark: the same back-to-back tcgen05.mma loop as umma_a_tmem.cu on ONE CTA pair and on ALL 148 SMs at once, with
// small-integer and with random bf16 operands, timed in SM cycles (clock64) and in nanoseconds (globaltimer).  An MMA takes 64
// (N = 128) / 128 (N = 256) CYCLES in every case; with random operands on the whole chip the SM clock drops (1845 -> 1610-1640 MHz
// within 2 ms; cuBLAS under sustained load: 1335 MHz, MEASURED_PEAKS.json), so the same MMAs take 1.15-1.4x the time.  That, not
// a pipeline stall, is the gap between the nominal dense bf16 rate and the 1659 TFLOP/s cuBLAS reaches here, and it is what the
// tensor phases of the codec kernels run at.
#include <cstdio>
#include "tc_common.cuh"
using namespace mapl::tc;

constexpr int kThreads = 320;      // warps 0-3: TMEM lanes (st / ld); warp 4: MMA issuer; warps 5-8: shared-memory traffic
constexpr int kACol = 256;         // A operand: columns [256, 384) = K 256 packed
constexpr int kNkb = 4;

__device__ int g_rand;
__device__ __forceinline__ float hashf(unsigned x) { x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16; return (float)(x & 0xffff) / 32768.f - 1.f; }
__device__ __forceinline__ float a_val(int m, int k) { return g_rand ? hashf(m * 4099u + k) : (float)((m * 7 + k * 3) % 13 - 6); }
__device__ __forceinline__ float b_val(int n, int k) { return g_rand ? hashf(n * 8191u + k + 77777u) : (float)((n * 5 + k * 11) % 9 - 4); }

__device__ __forceinline__ void umma_bf16_pair_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n"
      "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}

// mode 0: correctness (N = 128, K = 256); mode 1: timing
// CM / WT: a tcgen05.commit / a wait on an already completed mbarrier (+ fence) after every k-block of 4 MMAs: what the
// bookkeeping of a pipeline costs the issuing thread
template <int ts, int CM = 0, int WT = 0>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
k_ts(int mode, int N, int chunks, int with_ld, int with_smem, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sA = smem;                        // kNkb tiles [128 x 64] bf16 SW128 (the shared-memory A operand)
  uint8_t* sB = sA + kNkb * 16384;           // kNkb half tiles [N/2 x 64]
  uint8_t* sT = sB + kNkb * 16384;           // 32 KB of traffic scratch
  uint64_t* bar = reinterpret_cast<uint64_t*>(sT + 32768);
  uint32_t* slot = reinterpret_cast<uint32_t*>(bar + 4);
  volatile uint32_t* done = slot + 1;
  const uint32_t rank = cluster_ctarank();
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  // operands: row m of A = token row (rank * 128 + m); row n of this CTA's B half = n + rank * N/2
  for (int i = threadIdx.x; i < 128 * 32 * kNkb / 4; i += kThreads) {      // 16-byte pieces of A: (kb, row, chunk)
    const int kb = i / (128 * 8), row = (i / 8) % 128, ch = i % 8;
    uint32_t w[4];
    for (int e = 0; e < 4; ++e) {
      const int k = kb * 64 + ch * 8 + 2 * e;
      w[e] = pack_bf16x2(a_val(rank * 128 + row, k), a_val(rank * 128 + row, k + 1));
    }
    *reinterpret_cast<uint4*>(sA + kb * 16384 + sw128_offset(row, ch)) = make_uint4(w[0], w[1], w[2], w[3]);
  }
  for (int i = threadIdx.x; i < (N / 2) * 8 * kNkb; i += kThreads) {
    const int kb = i / ((N / 2) * 8), row = (i / 8) % (N / 2), ch = i % 8;
    uint32_t w[4];
    for (int e = 0; e < 4; ++e) {
      const int k = kb * 64 + ch * 8 + 2 * e;
      w[e] = pack_bf16x2(b_val(rank * (N / 2) + row, k), b_val(rank * (N / 2) + row, k + 1));
    }
    *reinterpret_cast<uint4*>(sB + kb * 16384 + sw128_offset(row, ch)) = make_uint4(w[0], w[1], w[2], w[3]);
  }
  if (threadIdx.x == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[2], 1); mbar_init(&bar[3], 1); *done = 0; fence_barrier_init(); }
  fence_proxy_async_smem();
  if (warp == 0) tmem_alloc_pair<512>(slot);
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem = *slot;
  if (warp < 4) {          // A into tensor memory: lane = row, column j of k-step s = (k = 16 s + 2j, 16 s + 2j + 1)
    const int row = warp * 32 + lane;
    for (int c0 = 0; c0 < kNkb * 32; c0 += 32) {
      uint32_t v[32];
#pragma unroll
      for (int j = 0; j < 32; ++j) v[j] = pack_bf16x2(a_val(rank * 128 + row, 2 * (c0 + j)), a_val(rank * 128 + row, 2 * (c0 + j) + 1));
      tmem_st32(tmem + ((uint32_t)(warp * 32) << 16) + kACol + c0, v);
    }
    tmem_st_wait();
  }
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  if (rank == 0 && threadIdx.x == 128) {
    const uint32_t idesc = make_idesc_bf16(256, N, false, false);
    const long long t0 = clock64();
    unsigned long long g0; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    for (int c = 0; c < chunks; ++c) {
      const uint32_t d = tmem + (N <= 128 ? (c & 1) * 128 : 0);
      for (int kb = 0; kb < kNkb; ++kb) {
        const uint32_t a = smem_u32(sA + kb * 16384), b = smem_u32(sB + kb * 16384);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (ts) umma_bf16_pair_ts(d, tmem + kACol + kb * 32 + k * 8, desc_kmajor_sw128(b + k * 32), idesc, (kb | k) != 0);
          else umma_bf16_pair(d, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc, (kb | k) != 0);
        }
        if (CM) umma_commit_pair(&bar[2]);
        if (WT) { mbar_wait(&bar[3], 1); tc_fence_after_sync(); }
      }
    }
    const long long t1 = clock64();
    umma_commit_pair(&bar[0]);
    mbar_wait(&bar[0], 0);
    const long long t2 = clock64();
    unsigned long long g1; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    out[0] = t1 - t0; out[1] = t2 - t0; out[12] = (long long)(g1 - g0);
    *done = 1;
  }
  if (mode == 1) {
    if (warp < 4 && with_ld) {             // read-out beside the MMAs (columns of the accumulator being written: timing only)
      uint32_t v[32]; uint32_t acc = 0; long long n = 0;
      while (!*done && n < 100000) {
        tmem_ld32(tmem + ((uint32_t)(warp * 32) << 16) + (n & 3) * 32, v);
        tmem_ld_wait();
        acc ^= v[0] ^ v[31]; ++n;
      }
      if (lane == 0 && rank == 0) out[4 + warp] = n * 32 * 32 * 4 + (acc == 0x12345u);
    }
    if (warp >= 5 && warp < 9 && with_smem) {      // conflict-free 16-byte stores + loads over 32 KB
      uint4 x = make_uint4(warp, lane, 0, 0); long long n = 0; uint32_t acc = 0;
      uint8_t* base = sT + (warp - 5) * 8192;
      while (!*done && n < 100000) {
#pragma unroll
        for (int i = 0; i < 8; ++i) *reinterpret_cast<uint4*>(base + i * 512 + lane * 16) = x;
#pragma unroll
        for (int i = 0; i < 8; ++i) acc ^= reinterpret_cast<volatile uint4*>(base + 4096 + i * 512 + lane * 16)->x;
        ++n;
      }
      if (lane == 0 && rank == 0) out[8 + warp - 5] = n * 16 * 512 + (acc == 0x12345u);
    }
  }
  if (rank == 1 && threadIdx.x == 128) { mbar_wait(&bar[0], 0); *done = 1; }
  __syncthreads();
  if (mode == 0 && warp < 4) {             // D[m][n] against integer arithmetic
    tc_fence_after_sync();
    const int m = rank * 128 + warp * 32 + lane;
    long long bad = 0;
    for (int c0 = 0; c0 < N; c0 += 32) {
      uint32_t v[32];
      tmem_ld32(tmem + ((uint32_t)(warp * 32) << 16) + c0, v);
      tmem_ld_wait();
      for (int j = 0; j < 32; ++j) {
        float ref = 0.f;
        for (int k = 0; k < 64 * kNkb; ++k) ref += a_val(m, k) * b_val(c0 + j, k);
        if (__uint_as_float(v[j]) != ref) ++bad;
      }
    }
    atomicAdd(reinterpret_cast<unsigned long long*>(&out[2]), (unsigned long long)bad);
  }
  tc_fence_before_sync();
  cluster_sync_all();
  if (warp == 0) { tc_fence_after_sync(); tmem_dealloc_pair<512>(tmem); }
}

int main() {
  long long* out; cudaMalloc(&out, 128);
  cudaFuncSetAttribute(k_ts<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  const size_t smem = 2 * kNkb * 16384 + 32768 + 1024 + 256;
  long long h[16];
  for (int rnd : {0, 1}) for (int grid : {2, 148}) for (int N : {128, 256}) {
    cudaMemcpyToSymbol(g_rand, &rnd, 4);
    const int chunks = 4000;
    for (int rep = 0; rep < 2; ++rep) { cudaMemset(out, 0, 128); k_ts<0><<<grid, kThreads, smem>>>(1, N, chunks, 0, 0, out); }
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("err %s\n", cudaGetErrorString(cudaGetLastError())); return 1; }
    cudaMemcpy(h, out, 128, cudaMemcpyDeviceToHost);
    printf("%s data, grid %3d CTAs, N %3d: %6.1f cycles, %6.2f ns per MMA -> %.0f MHz\n", rnd ? "random" : "small-int", grid, N, (double)h[1] / (chunks * kNkb * 4), (double)h[12] / (chunks * kNkb * 4), 1e3 * h[1] / (double)h[12]);
  }
  return 0;
}
