// tc_tile_ops.cuh -- the "token tile x d-chunks" streaming GEMM shared by decode and by the dH phase
// of backward:   Out[tile_m, d] = Aop[128, nkb*64] . W[d, nkb*64]^T
//   Aop   resident smem operand, nkb k-blocks of [128 x 64] bf16, K-major SW128
//   W     streamed by TMA in [128 x 64] tiles through a ring of b_stages
//   D     kAccStages x [128 lanes x 128 cols] fp32 in TMEM (MMA of chunk j+1 overlaps epilogue of j)
//   Out   bf16, through swizzled staging boxes and TMA stores
// Three roles, each called by the warp(s) that own it.
#pragma once
#include <stdlib.h>

#include "tc_common.cuh"

namespace mapl {
namespace tc {

constexpr int kChunkN = 128;                 // d-chunk width == UMMA N
constexpr int kTileBytes = 128 * 64 * 2;     // one [128 x 64] bf16 tile
constexpr int kAccStages = 4;
constexpr int kOutBufs = 4;

struct ChunkPipe {
  uint8_t* sA;        // resident A operand (nkb tiles)
  uint8_t* sB;        // ring (b_stages tiles)
  uint8_t* sOut;      // kOutBufs staging boxes
  uint64_t* b_full; uint64_t* b_empty;       // [b_stages]
  uint64_t* acc_full; uint64_t* acc_empty;   // [kAccStages]
  int nkb, nchunks, b_stages;
  uint32_t tmem_base;
};

// producer: one thread
__device__ __forceinline__ void chunk_produce(const ChunkPipe& c, const CUtensorMap* tmW) {
  int it = 0;
  for (int j = 0; j < c.nchunks; ++j)
    for (int kb = 0; kb < c.nkb; ++kb, ++it) {
      const int s = it % c.b_stages;
      mbar_wait(&c.b_empty[s], ((it / c.b_stages) & 1) ^ 1);
      mbar_arrive_expect_tx(&c.b_full[s], kTileBytes);
      tma_load_2d(c.sB + (size_t)s * kTileBytes, tmW, &c.b_full[s], kb * 64, j * kChunkN, kEvictLast);
    }
}

// MMA issuer: one thread; the A operand must already be visible to the async proxy
__device__ __forceinline__ void chunk_mma(const ChunkPipe& c) {
  const uint32_t idesc = make_idesc_bf16(128, kChunkN, false, false);
  int it = 0;
  for (int j = 0; j < c.nchunks; ++j) {
    const int as = j % kAccStages;
    mbar_wait(&c.acc_empty[as], ((j / kAccStages) & 1) ^ 1);
    tc_fence_after_sync();
    const uint32_t tmem_d = c.tmem_base + as * kChunkN;
    for (int kb = 0; kb < c.nkb; ++kb, ++it) {
      const int s = it % c.b_stages;
      mbar_wait(&c.b_full[s], (it / c.b_stages) & 1);
      tc_fence_after_sync();
      const uint32_t a = smem_u32(c.sA + (size_t)kb * kTileBytes), b = smem_u32(c.sB + (size_t)s * kTileBytes);
#pragma unroll
      for (int k = 0; k < 4; ++k)
        umma_bf16(tmem_d, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc, (kb | k) != 0);
      umma_commit(&c.b_empty[s]);
    }
    umma_commit(&c.acc_full[as]);
  }
}

// epilogue: the 4 warps with threadIdx.x in [64,192); row = TMEM lane = token row in the tile.
// Uses named barrier 1 (128 threads).  Thread 64 issues the TMA stores.
__device__ __forceinline__ void chunk_epilogue(const ChunkPipe& c, const CUtensorMap* tmO, int m0) {
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32, q = warp & 3, row = q * 32 + lane;
  for (int j = 0; j < c.nchunks; ++j) {
    const int as = j % kAccStages, ob = (j & 1) * 2;
    // only chunk j-1's store group may still be reading smem: the boxes of chunk j-2 are free
    if (threadIdx.x == 64) tma_store_wait_read<1>();
    asm volatile("bar.sync 1, 128;" ::: "memory");
    mbar_wait(&c.acc_full[as], (j / kAccStages) & 1);
    tc_fence_after_sync();
#pragma unroll
    for (int cc = 0; cc < kChunkN / 32; ++cc) {
      uint32_t v[32];
      tmem_ld32(c.tmem_base + ((uint32_t)(q * 32) << 16) + as * kChunkN + cc * 32, v);
      tmem_ld_wait();
      uint8_t* box = c.sOut + (size_t)(ob + cc / 2) * kTileBytes;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        uint4 o;
        o.x = pack_bf16x2(__uint_as_float(v[8 * i + 0]), __uint_as_float(v[8 * i + 1]));
        o.y = pack_bf16x2(__uint_as_float(v[8 * i + 2]), __uint_as_float(v[8 * i + 3]));
        o.z = pack_bf16x2(__uint_as_float(v[8 * i + 4]), __uint_as_float(v[8 * i + 5]));
        o.w = pack_bf16x2(__uint_as_float(v[8 * i + 6]), __uint_as_float(v[8 * i + 7]));
        *reinterpret_cast<uint4*>(box + sw128_offset(row, (cc & 1) * 4 + i)) = o;
      }
    }
    tc_fence_before_sync();
    __syncwarp();
    if (lane == 0) mbar_arrive(&c.acc_empty[as]);     // the TMEM stage may be overwritten
    fence_proxy_async_smem();
    asm volatile("bar.sync 1, 128;" ::: "memory");
    if (threadIdx.x == 64) {
      tma_store_2d(tmO, c.sOut + (size_t)ob * kTileBytes, j * kChunkN, m0);
      tma_store_2d(tmO, c.sOut + (size_t)(ob + 1) * kTileBytes, j * kChunkN + 64, m0);
      tma_store_commit();
    }
  }
  if (threadIdx.x == 64) tma_store_wait_all<0>();
}

__device__ __forceinline__ void chunk_init_barriers(const ChunkPipe& c) {
  for (int s = 0; s < c.b_stages; ++s) { mbar_init(&c.b_full[s], 1); mbar_init(&c.b_empty[s], 1); }
  for (int s = 0; s < kAccStages; ++s) { mbar_init(&c.acc_full[s], 1); mbar_init(&c.acc_empty[s], 4); }
}

// host: launch with programmatic dependent launch allowed (the kernels call griddepcontrol.wait
// before touching global memory)
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  static const bool pdl = getenv("MAPL_NO_PDL") == nullptr;     // debugging aid: plain stream order
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

}  // namespace tc
}  // namespace mapl
