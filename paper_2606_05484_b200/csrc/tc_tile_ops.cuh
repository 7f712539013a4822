// tc_tile_ops.cuh -- the "token tile x d-chunks" streaming GEMM shared by decode and by the dH phase
// of backward, run by a CTA PAIR (cluster of 2, tcgen05 cta_group::2):
//     Out[2 x 128 tokens, d] = Aop[2 x 128, nkb*64] . W[d, nkb*64]^T
//   Aop   resident smem operand of EACH CTA (its own 128 token rows), nkb k-blocks of [128 x 64]
//         bf16, K-major SW128
//   W     streamed by TMA through a ring of b_stages; per stage each CTA holds HALF of the
//         [128 x 64] tile (64 rows of W): the pair reads every W byte from L2 once, not twice
//   D     4 stages x [128 lanes x 128 cols] fp32 in each CTA's TMEM (MMA of chunk j+1 overlaps the
//         epilogue of chunk j); one M=256 UMMA per k-step, issued by the leader CTA (rank 0)
//   Out   bf16, through two swizzled staging boxes and TMA stores, each CTA its own rows.  (Direct
//         st.global from the row-per-thread register layout was measured 2x slower: 32 partial
//         sectors per instruction.)
// Barriers: b_full / acc_empty live in the leader (they collect arrivals from both CTAs);
// b_empty / acc_full exist in both CTAs and are signalled by multicast commits.
// Measured (profiles/): with the tensor pipe at ~75 % of nominal inside the chunk loop the MMA issue
// is the limiter there; the A-operand prologue of the callers is what remains exposed.
// Three roles, each called by the warp(s) that own it.
#pragma once
#include <stdlib.h>

#include "tc_common.cuh"

namespace mapl {
namespace tc {

constexpr int kChunkN = 256;                 // d-chunk width == UMMA N
constexpr int kTileBytes = 128 * 64 * 2;     // one [128 x 64] bf16 tile
constexpr int kHalfTileBytes = 64 * 64 * 2;  // the half of a W tile one CTA of the pair holds
constexpr int kAccStages = 2;
#ifndef MAPL_OUT_BUFS
#define MAPL_OUT_BUFS 4
#endif
constexpr int kOutBufs = MAPL_OUT_BUFS;      // [128 x 64] staging boxes: kOutBufs / 2 per column half (128 columns) of a chunk
constexpr int kBoxesPerHalf = kOutBufs / 2;
constexpr int kPipeThreads = 320;            // warp 0 TMA, warp 1 MMA, warps 2-9 epilogue

// Position in a ring of `size` stages, advanced without divisions: the TMA producer and MMA issuer loops run on ONE
// thread each, every instruction waits for the one before it (no other warp hides the latency), and an integer
// division by a run-time ring size is ~30 dependent instructions -- measured, the loops ran at ~600 cycles per
// iteration with `it % stages` / `it / stages`, against ~50 for the barrier + TMA instructions themselves.
struct RingPos {
  int st; uint32_t ph;       // stage, phase parity of the stage's current use (0 for the first pass)
  __device__ __forceinline__ RingPos() : st(0), ph(0) {}
  __device__ __forceinline__ void advance(int n, int size) {
    st += n;
    while (st >= size) { st -= size; ph ^= 1u; }
  }
  __device__ __forceinline__ void next(int size) {
    if (++st == size) { st = 0; ph ^= 1u; }
  }
};

struct ChunkPipe {
  uint8_t* sA;        // resident A operand (nkb tiles)
  uint8_t* sB;        // ring (b_stages half tiles)
  uint8_t* sOut;      // kOutBufs staging boxes
  uint64_t* b_full; uint64_t* b_empty;       // [b_stages]
  uint64_t* acc_full; uint64_t* acc_empty;   // [kAccStages]
  int nkb, nchunks, b_stages;
  uint32_t tmem_base, rank;   // rank = rank inside the pair
  PairPos pp;                 // pp.nq == 2: the W tiles are shared with the twin CTA of the other pair (multicast)
};

// producer: one thread in each CTA; tmW box = [128 / nq rows x 64 cols]
__device__ __forceinline__ void chunk_produce(const ChunkPipe& c, const CUtensorMap* tmW) {
  RingPos rp;
#ifdef MAPL_DBG
  long long w_empty = 0;
#endif
  for (int j = 0; j < c.nchunks; ++j)
    for (int kb = 0; kb < c.nkb; ++kb) {
#ifdef MAPL_DBG
      const long long t_a = clock64();
#endif
      mbar_wait(&c.b_empty[rp.st], rp.ph ^ 1u);
#ifdef MAPL_DBG
      w_empty += clock64() - t_a;
#endif
      if (c.rank == 0) mbar_arrive_expect_tx(&c.b_full[rp.st], 2 * kTileBytes);
      uint8_t* dst = c.sB + (size_t)rp.st * kTileBytes;
      const int row = j * kChunkN + (int)c.rank * (kChunkN / 2);
      if (c.pp.nq == 1) tma_load_2d_pair(dst, tmW, &c.b_full[rp.st], kb * 64, row, kEvictLast);
      else   // this CTA's half of the rows it holds, sent to itself and to its twin (tmW box: kChunkN / 4 rows)
        tma_load_2d_pair_mc(dst + (size_t)c.pp.q * (kTileBytes / 2), tmW, &c.b_full[rp.st], kb * 64, row + (int)c.pp.q * (kChunkN / 4),
                            c.pp.twin_mask, kEvictLast);
      rp.next(c.b_stages);
    }
#ifdef MAPL_DBG
  g_dbg[blockIdx.x * 64 + 62] = (unsigned long long)w_empty;      // cycles the producer waited for free ring slots
#endif
}

// MMA issuer: one thread of the LEADER CTA; the A operands of both CTAs must already be visible to
// the async proxy
__device__ __forceinline__ void chunk_mma(const ChunkPipe& c) {
  const uint32_t idesc = make_idesc_bf16(256, kChunkN, false, false);
  const uint32_t sA0 = smem_u32(c.sA), sB0 = smem_u32(c.sB);
  RingPos rp;
#ifdef MAPL_DBG
  long long w_acc = 0, w_full = 0, t_b;
#endif
  for (int j = 0; j < c.nchunks; ++j) {
    const int as = j % kAccStages;
#ifdef MAPL_DBG
    t_b = clock64();
#endif
    mbar_wait_cluster(&c.acc_empty[as], ((j / kAccStages) & 1) ^ 1);
#ifdef MAPL_DBG
    w_acc += clock64() - t_b;
#endif
    if (j < 16) DBGT(8 + j)
    tc_fence_after_sync();
    const uint32_t tmem_d = c.tmem_base + as * kChunkN;
    for (int kb = 0; kb < c.nkb; ++kb) {
#ifdef MAPL_DBG
      t_b = clock64();
#endif
      mbar_wait(&c.b_full[rp.st], rp.ph);
#ifdef MAPL_DBG
      w_full += clock64() - t_b;
#endif
      tc_fence_after_sync();
      const uint32_t a = sA0 + (uint32_t)kb * kTileBytes, b = sB0 + (uint32_t)rp.st * kTileBytes;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        umma_bf16_pair(tmem_d, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc, (kb | k) != 0);
      umma_commit_mask(&c.b_empty[rp.st], c.pp.all_mask);      // every CTA that writes into this stage (own pair + twins)
      rp.next(c.b_stages);
    }
    umma_commit_mask(&c.acc_full[as], c.pp.pair_mask);
    if (j < 16) DBGT(24 + j)
  }
#ifdef MAPL_DBG
  g_dbg[blockIdx.x * 64 + 60] = (unsigned long long)w_acc;       // cycles the MMA issuer waited for a free accumulator stage
  g_dbg[blockIdx.x * 64 + 61] = (unsigned long long)w_full;      // ... and for W tiles
#endif
}

// epilogue: the 8 warps with threadIdx.x in [64,320) of each CTA.  Warp w reads TMEM lane quarter
// q = w & 3 (row = token row in the tile) and column half h = (w - 2) / 4 of the chunk (128 columns), in two
// rounds of 64 columns = one [128 x 64] staging box each; the two halves run independently (named barriers 1
// and 2, 128 threads each; threads 64 and 192 issue the TMA stores of their boxes).
__device__ __forceinline__ void chunk_epilogue(const ChunkPipe& c, const CUtensorMap* tmO, int m0) {
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32, q = warp & 3, h = (warp - 2) >> 2, row = q * 32 + lane;
  const bool issuer = threadIdx.x == 64 + h * 128;
  for (int j = 0; j < c.nchunks; ++j) {
    const int as = j % kAccStages;
    mbar_wait(&c.acc_full[as], (j / kAccStages) & 1);
    if (threadIdx.x == 64 && j < 16) DBGT(40 + j)
    tc_fence_after_sync();
#pragma unroll
    for (int i = 0; i < kBoxesPerHalf; ++i) {
      uint8_t* box = c.sOut + (size_t)(h * kBoxesPerHalf + i) * kTileBytes;
      uint32_t v[2][32];
      const uint32_t taddr = c.tmem_base + ((uint32_t)(q * 32) << 16) + as * kChunkN + h * (kChunkN / 2) + i * 64;
      tmem_ld32(taddr, v[0]);
      tmem_ld32(taddr + 32, v[1]);
      tmem_ld_wait();
      if (i == kBoxesPerHalf - 1) {          // the whole stage is in registers / staged: it may be overwritten
        tc_fence_before_sync();
        __syncwarp();
        if (lane == 0) mbar_arrive_leader(&c.acc_empty[as]);
      }
      // the store that last used this box (the same round of chunk j - 1; in the first chunk whatever the caller
      // staged there) must have read it before it is rewritten: of this thread's bulk groups only the one committed
      // after it (the other round) may still be pending
      if (issuer) { if (j == 0) tma_store_wait_read<0>(); else tma_store_wait_read<kBoxesPerHalf - 1>(); }
      if (h == 0) asm volatile("bar.sync 1, 128;" ::: "memory"); else asm volatile("bar.sync 2, 128;" ::: "memory");
#pragma unroll
      for (int t = 0; t < 8; ++t) {
        const uint32_t* w = &v[t / 4][8 * (t % 4)];
        uint4 o;
        o.x = pack_bf16x2(__uint_as_float(w[0]), __uint_as_float(w[1]));
        o.y = pack_bf16x2(__uint_as_float(w[2]), __uint_as_float(w[3]));
        o.z = pack_bf16x2(__uint_as_float(w[4]), __uint_as_float(w[5]));
        o.w = pack_bf16x2(__uint_as_float(w[6]), __uint_as_float(w[7]));
        *reinterpret_cast<uint4*>(box + sw128_offset(row, t)) = o;
      }
      fence_proxy_async_smem();
      if (h == 0) asm volatile("bar.sync 1, 128;" ::: "memory"); else asm volatile("bar.sync 2, 128;" ::: "memory");
      if (issuer) {
        tma_store_2d_hint(tmO, box, j * kChunkN + h * (kChunkN / 2) + i * 64, m0, kEvictFirst);     // Hhat / dH: not read again by the codec
        tma_store_commit();
      }
    }
  }
  if (issuer) tma_store_wait_all<0>();
}

__device__ __forceinline__ void chunk_init_barriers(const ChunkPipe& c) {
  for (int s = 0; s < c.b_stages; ++s) { mbar_init(&c.b_full[s], 1); mbar_init(&c.b_empty[s], c.pp.nq); }
  for (int s = 0; s < kAccStages; ++s) { mbar_init(&c.acc_full[s], 1); mbar_init(&c.acc_empty[s], 16); }
}

// sA tiles [tile0, tile0 + width/64): row (q*32 + j) := bf16( sum_{l < nsrc} table[l*src_stride + idx_j[l]*width + :] ),
// zeros where idx < 0.  idx[] holds the indices of row q*32+lane.  One warp, convergent.  The loads
// of 8 row groups are issued back to back before any is consumed (the gathers are L2-latency bound).
// Two warps share a quarter: `part` (0/1) takes the first / second half of the row groups.
// gout != nullptr: the rows go to global memory instead (row (q*32 + j) at gout + j' * width, j' = q*32 + j;
// rows with idx < 0 are skipped), each row written as one coalesced segment.
template <int kBatch>
__device__ __forceinline__ void gather_sum_rows(uint8_t* sA, int tile0, int width, const float* __restrict__ table,
                                                long long src_stride, const int (&idx)[8], int nsrc, int q, int lane,
                                                int part, __nv_bfloat16* gout = nullptr) {
  const int lpr = width / 8, rpi = 32 / lpr, cc = lane % lpr, sub = lane / lpr;
  for (int it0 = part * (lpr / 2); it0 < (part + 1) * (lpr / 2); it0 += kBatch) {   // lpr = 32 / rpi row groups in all
    float acc[kBatch][8];
#pragma unroll
    for (int b = 0; b < kBatch; ++b)
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[b][j] = 0.f;
#pragma unroll
    for (int l = 0; l < 8; ++l) {
      if (l < nsrc) {
        float4 x[kBatch], y[kBatch];
#pragma unroll
        for (int b = 0; b < kBatch; ++b) {
          const int k = __shfl_sync(0xffffffffu, idx[l], (it0 + b) * rpi + sub);
          const float4* src = reinterpret_cast<const float4*>(table + l * src_stride + (long long)(k < 0 ? 0 : k) * width + cc * 8);
          x[b] = __ldg(src); y[b] = __ldg(src + 1);
          if (k < 0) { x[b] = make_float4(0.f, 0.f, 0.f, 0.f); y[b] = x[b]; }
        }
#pragma unroll
        for (int b = 0; b < kBatch; ++b) {
          acc[b][0] += x[b].x; acc[b][1] += x[b].y; acc[b][2] += x[b].z; acc[b][3] += x[b].w;
          acc[b][4] += y[b].x; acc[b][5] += y[b].y; acc[b][6] += y[b].z; acc[b][7] += y[b].w;
        }
      }
    }
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int rl = (it0 + b) * rpi + sub;
      const uint4 o = make_uint4(pack_bf16x2(acc[b][0], acc[b][1]), pack_bf16x2(acc[b][2], acc[b][3]),
                                 pack_bf16x2(acc[b][4], acc[b][5]), pack_bf16x2(acc[b][6], acc[b][7]));
      if (gout == nullptr) {
        *reinterpret_cast<uint4*>(sA + (size_t)(tile0 + cc / 8) * kTileBytes + sw128_offset(q * 32 + rl, cc % 8)) = o;
      } else if (__shfl_sync(0xffffffffu, idx[0], rl) >= 0) {
        *reinterpret_cast<uint4*>(gout + (long long)(q * 32 + rl) * width + cc * 8) = o;
      }
    }
  }
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

// same, as clusters of `cluster_x` CTAs (2: one CTA pair for cta_group::2; 4: two pairs sharing parameter tiles by
// multicast); grid.x must be a multiple of cluster_x
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_cluster(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                      unsigned cluster_x, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  static const bool pdl = getenv("MAPL_NO_PDL") == nullptr;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = cluster_x; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_pair(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                   Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  static const bool pdl = getenv("MAPL_NO_PDL") == nullptr;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = 2; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 2;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

}  // namespace tc
}  // namespace mapl
