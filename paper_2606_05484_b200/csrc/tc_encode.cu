// tc_encode.cu -- mapl_encode on the tensor cores (RVQ off): Z = H U  (Eq. 1, centred h).
//
// One CTA per token tile (tile_m <= 128 tokens, sized so the grid fills the 148 SMs evenly), CTAs in
// pairs (cluster of 2).  Warp 0 of each CTA streams its H tile [128 x 64] (HBM, evict-first) and HALF of the
// U^T tile [r/2 x 64] (L2-resident pack) through a TMA/mbarrier ring; one thread of the leader's warp 1
// issues tcgen05.mma cta_group::2 (M=256, N=r, K=16) into TMEM accumulators [128 lanes x r columns] of both
// CTAs; warps 2-5 read their TMEM lane quarter back (one token row per thread), round to bf16 and store
// the payload.
// Roofline: HBM (reads d*2 B/token, writes r*2 B/token).  Measured: 9.5 us at c1 of
// which ~5.5 us stream at 4.3 TB/s; the rest is prologue, first-stage latency and epilogue.
#include "profile.cuh"
#include "tc_codec.cuh"
#include "tc_common.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

constexpr int BM = 128, BK = 64, kThreads = 192;

constexpr int kATile = BM * BK * 2;   // 16 KB

// CTA pair: the two CTAs of a cluster own consecutive token tiles and run ONE M=256 MMA per k-step
// (cta_group::2).  Each CTA loads its own H tile and HALF of the U^T tile (r/2 rows), so the
// parameter stream from L2 is half that of two independent CTAs.  Only the leader (cluster rank 0)
// issues MMAs; its commits arrive on the barriers of both CTAs.
__global__ void __launch_bounds__(kThreads, 1)
k_tc_encode(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmW,
            __nv_bfloat16* __restrict__ Z, long long N, int d, int r, int stages, int tile_m,
            const int32_t* __restrict__ tok, const float* __restrict__ Tc) {   // Tc != NULL: z -= Tc[tok] (Eq. 1 centring)
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int b_tile = (r / 2) * BK * 2;                 // this CTA's half of the U^T tile
  const int stage_bytes = kATile + b_tile;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)stages * stage_bytes);
  uint64_t* empty = full + stages;
  uint64_t* accum_full = empty + stages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(accum_full + 1);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t rank = cluster_ctarank();
  const long long m0 = (long long)blockIdx.x * tile_m;
  const int nkb = d / BK;

  if (warp == 0) { DBG(0) }
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmH);
    tma_prefetch_desc(&tmW);
    for (int s = 0; s < stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_init(accum_full, 1);
    fence_barrier_init();
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"((uint32_t)r) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before_sync();
  cluster_sync_all();                                       // barriers of both CTAs initialised
  tc_fence_after_sync();
  const uint32_t tmem_d = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");       // everything below touches global memory
  if (warp == 0) { DBG(1) }

  if (warp == 0) {
    if (elect_one()) {
      const uint32_t tx = 2u * (uint32_t)(tile_m * 128 + b_tile);
      const int wrow = (int)rank * (r / 2);
      RingPos rp;                                    // no divisions in this one-thread loop (tc_tile_ops.cuh)
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(&empty[rp.st], rp.ph ^ 1u);
        if (rank == 0) mbar_arrive_expect_tx(&full[rp.st], tx);
        uint8_t* a = smem + (size_t)rp.st * stage_bytes;
        tma_load_2d_pair(a, &tmH, &full[rp.st], kb * BK, (int)m0, kEvictFirst);
        tma_load_2d_pair(a + kATile, &tmW, &full[rp.st], kb * BK, wrow, kEvictLast);
        rp.next(stages);
      }
    }
  } else if (warp == 1) {
    if (rank == 0 && elect_one()) {
      const uint32_t idesc = make_idesc_bf16(2 * BM, (uint32_t)r, false, false);
      const uint32_t smem0 = smem_u32(smem);
      RingPos rp;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(&full[rp.st], rp.ph);
#ifdef MAPL_DBG
        if (kb == 0) DBGT(2)
        if (kb == nkb - 1) DBGT(3)
#endif
        tc_fence_after_sync();
        const uint32_t a = smem0 + (uint32_t)rp.st * (uint32_t)stage_bytes;
        const uint32_t b = a + kATile;
#pragma unroll
        for (int k = 0; k < BK / 16; ++k)
          umma_bf16_pair(tmem_d, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc, (kb | k) != 0);
        umma_commit_pair(&empty[rp.st]);
        rp.next(stages);
      }
      umma_commit_pair(accum_full);
    }
  } else {
    const int q = warp & 3;                         // TMEM lane quarter this warp may read
    const int row = q * 32 + lane;
    const long long m = m0 + row;
    const bool live = row < tile_m && m < N;
    const float* trow = (Tc != nullptr && live) ? Tc + (long long)__ldg(tok + m) * r : nullptr;
    // centring rows are gathered (L2 latency): piece c+1 is in flight while piece c is consumed, piece 0 while the
    // MMAs still run
    float4 tcur[8], tnext[8];
    if (trow != nullptr) {
#pragma unroll
      for (int i = 0; i < 8; ++i) tcur[i] = __ldg(reinterpret_cast<const float4*>(trow) + i);
    }
    mbar_wait(accum_full, 0);
    if (warp == 2) { DBG(4) }
    tc_fence_after_sync();
    for (int c = 0; c < r / 32; ++c) {
      uint32_t v[32];
      tmem_ld32(tmem_d + ((uint32_t)(q * 32) << 16) + c * 32, v);
      if (trow != nullptr && c + 1 < r / 32) {
#pragma unroll
        for (int i = 0; i < 8; ++i) tnext[i] = __ldg(reinterpret_cast<const float4*>(trow + (c + 1) * 32) + i);
      }
      tmem_ld_wait();
      if (trow != nullptr) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          v[4 * i + 0] = __float_as_uint(__uint_as_float(v[4 * i + 0]) - tcur[i].x);
          v[4 * i + 1] = __float_as_uint(__uint_as_float(v[4 * i + 1]) - tcur[i].y);
          v[4 * i + 2] = __float_as_uint(__uint_as_float(v[4 * i + 2]) - tcur[i].z);
          v[4 * i + 3] = __float_as_uint(__uint_as_float(v[4 * i + 3]) - tcur[i].w);
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) tcur[i] = tnext[i];
      }
      if (live) {
        uint4* dst = reinterpret_cast<uint4*>(Z + m * r + c * 32);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          uint4 o;
          o.x = pack_bf16x2(__uint_as_float(v[8 * i + 0]), __uint_as_float(v[8 * i + 1]));
          o.y = pack_bf16x2(__uint_as_float(v[8 * i + 2]), __uint_as_float(v[8 * i + 3]));
          o.z = pack_bf16x2(__uint_as_float(v[8 * i + 4]), __uint_as_float(v[8 * i + 5]));
          o.w = pack_bf16x2(__uint_as_float(v[8 * i + 6]), __uint_as_float(v[8 * i + 7]));
          dst[i] = o;
        }
      }
    }
  }
  if (warp == 2) { DBG(5) }
  tc_fence_before_sync();
  cluster_sync_all();                                       // the peer may still signal our barriers / read our smem
  if (warp == 1) {
    tc_fence_after_sync();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"((uint32_t)r) : "memory");
  }
}

}  // namespace
}  // namespace mapl
MAPL_DBG_READER(mapl_debug_read_encode)
namespace mapl {

int tc_encode_rvq(const mapl_boundary_desc& d, const void* H, const float* codebooks, const TcPack& pk, void* Zq_out,
                  int32_t* codes_out, cudaStream_t st, const int32_t* tok, const float* Tc, void* ovf_ws);   // tc_encode_rvq.cu

int tc_encode(const mapl_boundary_desc& d, const void* H, const float* codebooks, const TcPack& pk, void* Zq_out,
              int32_t* codes_out, cudaStream_t st, const int32_t* tok, const float* Tc, void* ovf_ws) {
  if (!tc_shape_ok(d)) return MAPL_ERR_UNSUPPORTED;
  if (d.rvq_levels != 0) return tc_encode_rvq(d, H, codebooks, pk, Zq_out, codes_out, st, tok, Tc, ovf_ws);
  const int tile_m = tc_tile_m(d.n_tokens);
  CUtensorMap tmH, tmW;
  if (!make_tmap_bf16_2d(&tmH, H, (uint64_t)d.n_tokens, (uint64_t)d.d, (uint64_t)d.d, BK, (uint32_t)tile_m)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmW, pk.WB, (uint64_t)d.r, (uint64_t)d.d, (uint64_t)d.d, BK, (uint32_t)d.r / 2)) return MAPL_ERR_CUDA;
  const int stage_bytes = kATile + (d.r / 2) * BK * 2;
  int stages = (200 * 1024) / stage_bytes;
  if (stages > 8) stages = 8;
  if (stages > d.d / BK) stages = d.d / BK;
  const size_t smem = (size_t)stages * stage_bytes + 1024 + 256;
  MAPL_SMEM_OPT_IN(k_tc_encode, 227 * 1024);
  const unsigned tiles = ((unsigned)((d.n_tokens + tile_m - 1) / tile_m) + 1u) & ~1u;   // whole CTA pairs
  KernelScope ks(KID_TC_ENCODE, st);
  MAPL_CUDA_CHECK(launch_pdl_pair(k_tc_encode, dim3(tiles), dim3(kThreads), smem, st, tmH, tmW,
                             reinterpret_cast<__nv_bfloat16*>(Zq_out), d.n_tokens, d.d, d.r, stages, tile_m, tok, Tc));
  return MAPL_OK;
}

}  // namespace mapl
