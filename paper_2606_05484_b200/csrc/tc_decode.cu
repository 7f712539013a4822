// tc_decode.cu -- mapl_decode on the tensor cores:  Hhat = [Zhat | A[tok]] . [U | B^T]^T
// (Eq. 2 with the factorised anchor of PAPER.md:106 Eq. 3 folded in as extra K columns).
//
// One CTA per token tile (tile_m <= 128 tokens, sized so the grid fills the 148 SMs evenly); CTAs
// work in pairs (cluster of 2, cta_group::2 MMAs of M = 256, see tc_tile_ops.cuh).
//   A operand  [128 x Kc] bf16, K-major SW128, resident for the CTA's lifetime:
//                columns [0,r): Zhat -- TMA from the wire payload, or dequantised from the RVQ
//                codes by the epilogue warps (gather-sum of codewords, fp32, rounded once);
//                columns [r,Kc): rows A[tok] gathered from the fp32 table by the epilogue warps.
//   B operand  Wd pack [d, Kc] bf16 streamed through a TMA/mbarrier ring, half a [128 x 64] tile per CTA.
//   D, epilogue: see tc_tile_ops.cuh.
// Roofline: HBM (writes d*2 B/token).
#include "profile.cuh"
#include "tc_codec.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

constexpr int kThreads = kPipeThreads;

struct DecodeParams {
  const int32_t* codes; const float* codebooks;   // RVQ dequant (codes != nullptr)
  const int32_t* tok; const float* A;             // anchor gather (tok != nullptr)
  long long N;
  int d, r, ra, L, K;
  int tile_m, b_stages, z_from_tma, nq;
};

__global__ void __launch_bounds__(kThreads, 1)
k_tc_decode(const __grid_constant__ CUtensorMap tmZ, const __grid_constant__ CUtensorMap tmW,
            const __grid_constant__ CUtensorMap tmO, const DecodeParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  ChunkPipe c;
  c.nkb = (p.r + p.ra) / 64; c.nchunks = p.d / kChunkN; c.b_stages = p.b_stages;
  c.pp = pair_pos((uint32_t)p.nq);
  c.rank = c.pp.pr;
  c.sA = smem;
  c.sOut = c.sA + (size_t)c.nkb * kTileBytes;
  c.sB = c.sOut + (size_t)kOutBufs * kTileBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(c.sB + (size_t)p.b_stages * kTileBytes);
  c.b_full = bars; c.b_empty = c.b_full + p.b_stages;
  c.acc_full = c.b_empty + p.b_stages; c.acc_empty = c.acc_full + kAccStages;
  uint64_t* a_full = c.acc_empty + kAccStages;         // leader's: A operands of both CTAs are in place
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(a_full + 1);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const long long m0 = (long long)blockIdx.x * p.tile_m;

  if (warp == 0) DBG(0)
#ifdef MAPL_DBG
  if (threadIdx.x == 0) { g_dbg[blockIdx.x * 64 + 5] = 0; g_dbg[blockIdx.x * 64 + 6] = 0; }
#endif
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmZ); tma_prefetch_desc(&tmW); tma_prefetch_desc(&tmO);
    chunk_init_barriers(c);
    mbar_init(a_full, 1 + 16);                // leader's producer (expect_tx) + the epilogue warps of both CTAs
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(tmem_slot);
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  c.tmem_base = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");       // everything below touches global memory
  if (warp == 0) DBG(1)

  if (warp == 0) {
    if (elect_one()) {
      if (p.z_from_tma) {
        if (c.rank == 0) mbar_arrive_expect_tx(a_full, 2u * (uint32_t)((p.r / 64) * p.tile_m * 128));
        for (int kb = 0; kb < p.r / 64; ++kb)
          tma_load_2d_pair(c.sA + (size_t)kb * kTileBytes, &tmZ, a_full, kb * 64, (int)m0, kEvictFirst);
      } else if (c.rank == 0) {
        mbar_arrive(a_full);
      }
      chunk_produce(c, &tmW);
    }
  } else if (warp == 1) {
    if (c.rank == 0 && elect_one()) {
      mbar_wait_cluster(a_full, 0);
      DBGT(2)
      tc_fence_after_sync();
      chunk_mma(c);
    }
  } else {
    const int q = warp & 3, part = (warp - 2) >> 2;
    const int row = q * 32 + lane;                      // token row inside the tile == TMEM lane
    const long long m = m0 + row;
    const bool live = row < p.tile_m && m < p.N;
    // ---- A operand columns produced by the warps: dequantised zhat and gathered anchor rows.
    // Warp-cooperative: r/8 (ra/8) lanes share one row, each lane one 16-byte bf16 chunk, so a
    // table row is read as one coalesced segment; this lane keeps the indices of row q*32+lane.
    if (!p.z_from_tma) {
      int idx[8];
#pragma unroll
      for (int l = 0; l < 8; ++l) idx[l] = (live && l < p.L) ? __ldg(p.codes + m * p.L + l) : -1;
      if (p.r >= 128) gather_sum_rows<8>(c.sA, 0, p.r, p.codebooks, (long long)p.K * p.r, idx, p.L, q, lane, part);
      else gather_sum_rows<4>(c.sA, 0, p.r, p.codebooks, (long long)p.K * p.r, idx, p.L, q, lane, part);
    }
    if (p.ra > 0) {
      int idx[8];
#pragma unroll
      for (int l = 0; l < 8; ++l) idx[l] = -1;
      idx[0] = live ? __ldg(p.tok + m) : -1;
      if (p.ra >= 128) gather_sum_rows<8>(c.sA, p.r / 64, p.ra, p.A, 0, idx, 1, q, lane, part);
      else gather_sum_rows<4>(c.sA, p.r / 64, p.ra, p.A, 0, idx, 1, q, lane, part);
    }
    fence_proxy_async_smem();
    __syncwarp();
    if (warp == 2) DBG(3)
    if (lane == 0) mbar_arrive_leader(a_full);
    chunk_epilogue(c, &tmO, (int)m0);
  }
  if (warp == 2) DBG(4)
  tc_fence_before_sync();
  cluster_sync_all();                       // the peer may still signal our barriers / its MMAs read our smem
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc_pair<512>(c.tmem_base);
  }
}

}  // namespace
}  // namespace mapl
MAPL_DBG_READER(mapl_debug_read_decode)
namespace mapl {

int tc_decode(const mapl_boundary_desc& d, const void* Z, const int32_t* codes, const float* codebooks,
              const int32_t* tok, const float* A, const TcPack& pk, void* Hhat_out, cudaStream_t st) {
  if (!tc_shape_ok(d)) return MAPL_ERR_UNSUPPORTED;
  const int ra = d.anchor_rank, kc = d.r + ra, nkb = kc / 64;
  DecodeParams p;
  p.codes = codes; p.codebooks = codebooks; p.tok = ra ? tok : nullptr; p.A = A;
  p.N = d.n_tokens; p.d = d.d; p.r = d.r; p.ra = ra; p.L = d.rvq_levels; p.K = d.rvq_k;
  p.nq = tc_pairs_per_cluster();
  p.tile_m = p.nq == 2 ? tc_tile_m4(d.n_tokens) : tc_tile_m(d.n_tokens);
  p.z_from_tma = codes ? 0 : 1;
  const size_t fixed = (size_t)(nkb + kOutBufs) * kTileBytes + 1024 + 512;
  p.b_stages = (int)((227 * 1024 - fixed) / kTileBytes);
  if (p.b_stages > 16) p.b_stages = 16;
  if (p.b_stages < 2) return MAPL_ERR_UNSUPPORTED;
  const size_t smem = fixed + (size_t)p.b_stages * kTileBytes;
  CUtensorMap tmZ, tmW, tmO;
  // Z: [N, r]; when zhat comes from codes the map is unused but must be valid: point it at the pack
  const void* zbase = codes ? (const void*)pk.Wd : Z;
  if (!make_tmap_bf16_2d(&tmZ, zbase, codes ? (uint64_t)d.d : (uint64_t)d.n_tokens, codes ? (uint64_t)kc : (uint64_t)d.r,
                         codes ? (uint64_t)kc : (uint64_t)d.r, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmW, pk.Wd, (uint64_t)d.d, (uint64_t)kc, (uint64_t)kc, 64, (uint32_t)(kChunkN / 2 / p.nq))) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmO, Hhat_out, (uint64_t)d.n_tokens, (uint64_t)d.d, (uint64_t)d.d, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
  MAPL_SMEM_OPT_IN(k_tc_decode, 227 * 1024);
  const unsigned cl = 2u * (unsigned)p.nq;
  const unsigned tiles = ((unsigned)((d.n_tokens + p.tile_m - 1) / p.tile_m) + cl - 1u) / cl * cl;   // whole clusters
  KernelScope ks(KID_TC_DECODE, st);
  MAPL_CUDA_CHECK(launch_pdl_cluster(k_tc_decode, dim3(tiles), dim3(kThreads), smem, st, cl, tmZ, tmW, tmO, p));
  return MAPL_OK;
}

}  // namespace mapl
