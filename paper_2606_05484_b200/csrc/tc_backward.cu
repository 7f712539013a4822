// tc_backward.cu -- mapl_codec_backward on the tensor cores (STE = S7).
//
// k_tc_bwd_gz   one CTA per token tile, CTAs in pairs (cta_group::2, M = 256: every parameter byte is
//               read from L2 once per pair); two phases over one read of g:
//     phase 1   [gz | gA] = g . [U | B^T]         K = d, streamed through a TMA ring
//               epilogue (8 warps): gz -> bf16 -> swizzled smem tiles that are both the A operand of
//               phase 2 and the source of the TMA store to gz_out (the backward wire payload);
//               gA rows -> fp32 scratch [N,ra] (TMA stores from the staging boxes).
//               With RVQ the same warps first dequantise the tile's codes into the bf16 Zhat
//               operand of k_tc_bwd_du (hidden under the g stream).
//     phase 2   dH = gz . U^T                     the chunk pipeline of tc_tile_ops.cuh
//               While phase 1 streams, the epilogue warps zero dU / dA / dB (overwrite mode): no
//               separate memset launches.
// k_tc_bwd_du   dU[d-tile, :] += sum over a token range of  g^T Zhat + H^T gz.  Both operands are
//               MN-major (tokens are the contraction index): TMA boxes [64 tokens x 64 cols]
//               are used as they land.  Split over token ranges; the fp32 tile is added to dU by TMA reductions.
//               r >= 128: CTA pairs (two d-tiles, M = 256, half of the Zhat / gz columns per CTA).
//               Its main loop streams g and H at 6.2 TB/s (measured, c1).
//               While the MMAs run, the epilogue warps scatter-add the gA rows into dA[tok]:
//               per 128-token block the ids are ranked in shared memory and rows of equal id are
//               summed in registers (Zipf ids: the hottest id owns ~14 % of all rows), then one
//               red.global.add row per distinct id leaves the CTA.
// Roofline: HBM at configs 1-2 (g, H read; dH written), tensor at config 3.
#include "profile.cuh"
#include "tc_codec.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

constexpr int kThreads = kPipeThreads;   // k_tc_bwd_gz: warp 0 TMA, warp 1 MMA, warps 2-9 epilogue
constexpr int kThreadsDu = 192;

__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// ---------------------------------------------------------------- gz / dA / dH
struct BwdGzParams {
  float* gA; __nv_bfloat16* gz_out;
  float* z0; long long n0;      // overwrite mode: fp32 arrays to zero (element counts, multiples of 4)
  float* z1; long long n1;
  float* z2; long long n2;
  long long N;
  int d, r, ra, tile_m;
  int stages1, stage1_bytes, b_stages, do_dh, ga_tma, nq;
  const int32_t* codes; const float* codebooks; __nv_bfloat16* zhat_out; int L, K;   // RVQ: zhat for k_tc_bwd_du
};

__global__ void __launch_bounds__(kThreads, 1)
k_tc_bwd_gz(const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmWu,
            const __grid_constant__ CUtensorMap tmWb, const __grid_constant__ CUtensorMap tmWd,
            const __grid_constant__ CUtensorMap tmO, const __grid_constant__ CUtensorMap tmGz,
            const __grid_constant__ CUtensorMap tmGA, const BwdGzParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int kc = p.r + p.ra, nkb1 = p.d / 64;
  // region R: phase 1 ring  |aliased with|  phase 2 gz operand + W ring
  const size_t ring1 = (size_t)p.stages1 * p.stage1_bytes;
  const size_t ring2 = (size_t)(p.r / 64) * kTileBytes + (size_t)p.b_stages * kTileBytes;
  const size_t regionR = ring1 > ring2 ? ring1 : ring2;
  ChunkPipe c;
  c.nkb = p.r / 64; c.nchunks = p.d / kChunkN; c.b_stages = p.b_stages;
  c.pp = pair_pos((uint32_t)p.nq);
  c.rank = c.pp.pr;
  c.sA = smem;
  c.sB = smem + (size_t)(p.r / 64) * kTileBytes;
  c.sOut = smem + regionR;
  uint64_t* bars = reinterpret_cast<uint64_t*>(c.sOut + (size_t)kOutBufs * kTileBytes);
  c.b_full = bars; c.b_empty = c.b_full + p.b_stages;
  c.acc_full = c.b_empty + p.b_stages; c.acc_empty = c.acc_full + kAccStages;
  uint64_t* s1_full = c.acc_empty + kAccStages;
  uint64_t* s1_empty = s1_full + p.stages1;
  uint64_t* acc1_full = s1_empty + p.stages1;
  uint64_t* gz_full = acc1_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(gz_full + 1);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const long long m0 = (long long)blockIdx.x * p.tile_m;

  if (warp == 0) DBG(56)
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmG); tma_prefetch_desc(&tmWu); tma_prefetch_desc(&tmWb);
    tma_prefetch_desc(&tmWd); tma_prefetch_desc(&tmO); tma_prefetch_desc(&tmGz); tma_prefetch_desc(&tmGA);
    chunk_init_barriers(c);
    for (int s = 0; s < p.stages1; ++s) { mbar_init(&s1_full[s], 1); mbar_init(&s1_empty[s], p.nq); }
    mbar_init(acc1_full, 1);
    mbar_init(gz_full, 16);                   // leader's: the epilogue warps of both CTAs
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(tmem_slot);
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  c.tmem_base = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (warp == 0) DBG(57)

  if (warp == 0) {
    if (elect_one()) {
      const uint32_t bytes = (uint32_t)(p.tile_m * 128 + kc * 64);   // per CTA: g tile + half of the [U^T;B] rows
      RingPos rp;                                    // no divisions in this one-thread loop (tc_tile_ops.cuh)
      for (int kb = 0; kb < nkb1; ++kb, rp.next(p.stages1)) {
        const int s = rp.st;
        mbar_wait(&s1_empty[s], rp.ph ^ 1u);
        if (c.rank == 0) mbar_arrive_expect_tx(&s1_full[s], 2 * bytes);
        uint8_t* a = smem + (size_t)s * p.stage1_bytes;
        tma_load_2d_pair(a, &tmG, &s1_full[s], kb * 64, (int)m0, kEvictLast);   // g is read again by k_tc_bwd_du
        if (p.nq == 1) {
          tma_load_2d_pair(a + kTileBytes, &tmWu, &s1_full[s], kb * 64, (int)c.rank * (p.r / 2), kEvictLast);
          if (p.ra) tma_load_2d_pair(a + kTileBytes + p.r * 64, &tmWb, &s1_full[s], kb * 64, p.r + (int)c.rank * (p.ra / 2), kEvictLast);
        } else {   // the parameter rows this CTA holds: half loaded here, half by the twin CTA of the other pair (multicast)
          const int q = (int)c.pp.q;
          tma_load_2d_pair_mc(a + kTileBytes + q * (p.r * 32), &tmWu, &s1_full[s], kb * 64, (int)c.rank * (p.r / 2) + q * (p.r / 4),
                              c.pp.twin_mask, kEvictLast);
          if (p.ra)
            tma_load_2d_pair_mc(a + kTileBytes + p.r * 64 + q * (p.ra * 32), &tmWb, &s1_full[s], kb * 64,
                                p.r + (int)c.rank * (p.ra / 2) + q * (p.ra / 4), c.pp.twin_mask, kEvictLast);
        }
      }
      if (p.do_dh) {
        mbar_wait(acc1_full, 0);        // phase 1 MMAs have consumed the ring: region R may be reused
        chunk_produce(c, &tmWd);
      }
    }
  } else if (warp == 1) {
    if (c.rank == 0 && elect_one()) {
      const uint32_t idesc_u = make_idesc_bf16(256, (uint32_t)p.r, false, false);
      const uint32_t idesc_b = make_idesc_bf16(256, (uint32_t)(p.ra ? p.ra : 64), false, false);
      const uint32_t smem0 = smem_u32(smem);
      RingPos rp;
      for (int kb = 0; kb < nkb1; ++kb, rp.next(p.stages1)) {
        const int s = rp.st;
        mbar_wait(&s1_full[s], rp.ph);
        tc_fence_after_sync();
        const uint32_t a = smem0 + (uint32_t)s * (uint32_t)p.stage1_bytes;
        const uint32_t bu = a + kTileBytes, bb = bu + p.r * 64;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint64_t da = desc_kmajor_sw128(a + k * 32);
          umma_bf16_pair(c.tmem_base, da, desc_kmajor_sw128(bu + k * 32), idesc_u, (kb | k) != 0);
          if (p.ra) umma_bf16_pair(c.tmem_base + p.r, da, desc_kmajor_sw128(bb + k * 32), idesc_b, (kb | k) != 0);
        }
        umma_commit_mask(&s1_empty[s], c.pp.all_mask);
      }
      umma_commit_mask(acc1_full, c.pp.pair_mask);
      if (p.do_dh) {
        mbar_wait_cluster(gz_full, 0);          // gz operand written and the phase 1 accumulator drained
        tc_fence_after_sync();
        chunk_mma(c);
      }
    }
  } else {
    const int q = warp & 3, half = (warp - 2) >> 2, row = q * 32 + lane;   // two warps per TMEM lane quarter
    const long long m = m0 + row;
    const bool live = row < p.tile_m && m < p.N;
    const uint32_t tmem_row = c.tmem_base + ((uint32_t)(q * 32) << 16);
    {   // overwrite mode: this CTA's slice of dU / dA / dB := 0 while phase 1 streams
      const int et = threadIdx.x - 64;
      const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
      float* zp[3] = {p.z0, p.z1, p.z2};
      const long long zn[3] = {p.n0, p.n1, p.n2};
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        if (zp[a] == nullptr) continue;
        const long long nv = zn[a] / 4, per = (nv + gridDim.x - 1) / gridDim.x;
        const long long lo = per * blockIdx.x, hi = lo + per < nv ? lo + per : nv;
        for (long long i = lo + et; i < hi; i += 256) reinterpret_cast<float4*>(zp[a])[i] = zero;
      }
    }
    if (p.codes != nullptr) {   // RVQ: dequantise this tile's codes into the bf16 zhat operand of k_tc_bwd_du while g streams
      int idx[8];
#pragma unroll
      for (int l = 0; l < 8; ++l) idx[l] = (live && l < p.L) ? __ldg(p.codes + m * p.L + l) : -1;
      __nv_bfloat16* gout = p.zhat_out + m0 * p.r;
      if (p.r >= 128) gather_sum_rows<8>(nullptr, 0, p.r, p.codebooks, (long long)p.K * p.r, idx, p.L, q, lane, half, gout);
      else gather_sum_rows<4>(nullptr, 0, p.r, p.codebooks, (long long)p.K * p.r, idx, p.L, q, lane, half, gout);
    }
    mbar_wait(acc1_full, 0);
    if (warp == 2) DBG(58)
    tc_fence_after_sync();
    // 32-column pieces alternate between the two warps; r >= 128: two pieces per TMEM wait.
    // The bf16 gz tile is both the A operand of phase 2 and the source of the TMA store to gz_out.
    auto put_piece = [&](const uint32_t (&v)[32], int cc) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        uint4 o;
        o.x = pack_bf16x2(__uint_as_float(v[8 * i + 0]), __uint_as_float(v[8 * i + 1]));
        o.y = pack_bf16x2(__uint_as_float(v[8 * i + 2]), __uint_as_float(v[8 * i + 3]));
        o.z = pack_bf16x2(__uint_as_float(v[8 * i + 4]), __uint_as_float(v[8 * i + 5]));
        o.w = pack_bf16x2(__uint_as_float(v[8 * i + 6]), __uint_as_float(v[8 * i + 7]));
        *reinterpret_cast<uint4*>(c.sA + (size_t)(cc / 2) * kTileBytes + sw128_offset(row, (cc & 1) * 4 + i)) = o;
      }
    };
    if (p.r == 64) {
      uint32_t v[32];
      tmem_ld32(tmem_row + half * 32, v);
      tmem_ld_wait();
      put_piece(v, half);
    } else {
      for (int cc = half; cc < p.r / 32; cc += 4) {       // r is 128 or 256 here (tc_shape_ok)
        uint32_t v0[32], v1[32];
        tmem_ld32(tmem_row + cc * 32, v0);
        tmem_ld32(tmem_row + (cc + 2) * 32, v1);
        tmem_ld_wait();
        put_piece(v0, cc);
        put_piece(v1, cc + 2);
      }
    }
    // gA staging: the ra / 32 pieces spread over the kOutBufs boxes (ra = 64: boxes 0 and 2, ra = 128: all four), so that
    // thread 64 stores from its own boxes [0, kBoxesPerHalf) and thread 192 from the rest (chunk_epilogue reuses them)
    const int ga_step = p.ra ? kOutBufs / (p.ra / 32) : 1;
    if (p.ra) {
      float4* dst = reinterpret_cast<float4*>(p.gA + (live ? m : 0) * p.ra);
      for (int cc = half; cc < p.ra / 32; cc += 2) {
        uint32_t v[32];
        tmem_ld32(tmem_row + p.r + cc * 32, v);
        tmem_ld_wait();
        if (p.ga_tma) {          // piece cc = [128 rows x 32 floats] -> staging box cc * ga_step, swizzled, stored by TMA below
#pragma unroll
          for (int i = 0; i < 8; ++i)
            *reinterpret_cast<float4*>(c.sOut + (size_t)cc * ga_step * kTileBytes + sw128_offset(row, i)) =
                make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]),
                            __uint_as_float(v[4 * i + 3]));
        } else if (live) {
#pragma unroll
          for (int i = 0; i < 8; ++i)
            dst[cc * 8 + i] = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]),
                                          __uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3]));
        }
      }
    }
    if (warp == 2) DBG(61)
    fence_proxy_async_smem();
    if (p.do_dh) {                    // release the phase-2 MMAs first: the TMA stores below only read the same tiles
      tc_fence_before_sync();
      __syncwarp();
      if (warp == 2) DBG(59)
      if (lane == 0) mbar_arrive_leader(gz_full);
    }
    asm volatile("bar.sync 3, 256;" ::: "memory");
    if (warp == 2) DBG(62)
    if (threadIdx.x == 64) {
      for (int kb = 0; kb < p.r / 64; ++kb) tma_store_2d(&tmGz, c.sA + (size_t)kb * kTileBytes, kb * 64, (int)m0);
      if (p.ga_tma)
        for (int cc = 0; cc * ga_step < kBoxesPerHalf; ++cc)
          tma_store_2d(&tmGA, c.sOut + (size_t)cc * ga_step * kTileBytes, cc * 32, (int)m0);
      tma_store_commit();
      if (!p.do_dh) tma_store_wait_all<0>();
    }
    if (threadIdx.x == 192 && p.ga_tma) {
      for (int cc = 0; cc < p.ra / 32; ++cc)
        if (cc * ga_step >= kBoxesPerHalf) tma_store_2d(&tmGA, c.sOut + (size_t)cc * ga_step * kTileBytes, cc * 32, (int)m0);
      tma_store_commit();
      if (!p.do_dh) tma_store_wait_all<0>();
    }
    if (p.do_dh) {
      if (warp == 2) DBG(63)
      chunk_epilogue(c, &tmO, (int)m0);
    }
    if (warp == 2) DBG(60)
  }
  tc_fence_before_sync();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc_pair<512>(c.tmem_base);
  }
}

// ---------------------------------------------------------------- dU
struct BwdDuParams {
  float* dU;
  long long N;
  int d, r, n_src, stages, item_bytes, blocks_per_split, n_blocks;
  const int32_t* tok; const float* gA; float* dA;   // anchor-gradient scatter (tok == nullptr: none)
  int ra;
};

// dA[tok_n, :] += gA[n, :] for the 128-token blocks this CTA owns; called by the 128 epilogue threads.
// Per block: all gA rows are staged in shared memory (every load in flight before the first store),
// the token ids are ranked (counting sort, 128 broadcast reads per thread), then the thread that holds
// the FIRST sorted position of an id sums the rows of that id in registers and issues one
// red.global.add.v4 row: no shared-memory atomics, and a hot Zipf id costs one global row per
// block instead of one per occurrence.
template <int kRa>
__device__ __forceinline__ void scatter_gA_t(const BwdDuParams& p, float* sG, int* sTok, int cta, int n_ctas) {
  constexpr int kPitch = kRa + 4, kVpr = kRa / 4, kLoads = kVpr;      // 128 rows * kVpr float4 / 128 threads
  const int et = threadIdx.x - 64;
  int* sSorted = sTok + 128;      // token id at each sorted position
  int* sOrder = sTok + 256;       // source row of each sorted position
  for (long long base = (long long)cta * 128; base < p.N; base += (long long)n_ctas * 128) {
    const int cnt = (int)(p.N - base < 128 ? p.N - base : 128);
    const float4* src = reinterpret_cast<const float4*>(p.gA + base * kRa);
    const int my = et < cnt ? __ldg(p.tok + base + et) : 0x7fffffff;
    float4 x[kLoads];
#pragma unroll
    for (int i = 0; i < kLoads; ++i) {
      const int f = et + i * 128;                     // float4 index inside the block
      x[i] = f < cnt * kVpr ? __ldg(src + f) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    sTok[et] = my;
#pragma unroll
    for (int i = 0; i < kLoads; ++i) {
      const int f = et + i * 128;
      *reinterpret_cast<float4*>(sG + (f / kVpr) * kPitch + (f % kVpr) * 4) = x[i];
    }
    asm volatile("bar.sync 1, 128;" ::: "memory");
    int rank = 0;
#pragma unroll 8
    for (int j = 0; j < 128; ++j) {
      const int t = sTok[j];
      rank += (t < my || (t == my && j < et)) ? 1 : 0;
    }
    sSorted[rank] = my;
    sOrder[rank] = et;
    asm volatile("bar.sync 1, 128;" ::: "memory");
    // thread et owns sorted position et
    const int id = sSorted[et];
    const bool head = id != 0x7fffffff && (et == 0 || sSorted[et - 1] != id);
    if (head) {
      float4 acc[kVpr];
      const float4* r0 = reinterpret_cast<const float4*>(sG + sOrder[et] * kPitch);
#pragma unroll
      for (int c = 0; c < kVpr; ++c) acc[c] = r0[c];
      for (int pos = et + 1; pos < 128 && sSorted[pos] == id; ++pos) {
        const float4* rr = reinterpret_cast<const float4*>(sG + sOrder[pos] * kPitch);
#pragma unroll
        for (int c = 0; c < kVpr; ++c) { const float4 v = rr[c]; acc[c].x += v.x; acc[c].y += v.y; acc[c].z += v.z; acc[c].w += v.w; }
      }
      float* dst = p.dA + (long long)id * kRa;
#pragma unroll
      for (int c = 0; c < kVpr; ++c) red_add_v4(dst + c * 4, acc[c].x, acc[c].y, acc[c].z, acc[c].w);
    }
    asm volatile("bar.sync 1, 128;" ::: "memory");
  }
}
__device__ __forceinline__ void scatter_gA(const BwdDuParams& p, float* sG, int* sTok, int cta, int n_ctas) {
  if (p.ra == 64) scatter_gA_t<64>(p, sG, sTok, cta, n_ctas); else scatter_gA_t<128>(p, sG, sTok, cta, n_ctas);
}

// kPair: two CTAs of a cluster own adjacent 128-row tiles of dU and the same token range; one M=256
// cta_group::2 MMA per 16 tokens, each CTA loading its own g/H boxes and HALF of the Zhat/gz columns
// (r >= 128).  !kPair: one CTA per d-tile (r == 64, where half an operand row is below the 128-byte
// swizzle span).
template <bool kPair>
__global__ void __launch_bounds__(kThreadsDu, 1)
k_tc_bwd_du(const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmZ,
            const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmGz,
            const __grid_constant__ CUtensorMap tmDU, const BwdDuParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)p.stages * p.item_bytes);
  uint64_t* empty = full + p.stages;
  uint64_t* acc_full = empty + p.stages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_full + 1);
  float* sG = reinterpret_cast<float*>(smem + (size_t)p.stages * p.item_bytes + 512);   // [128][ra+4]
  int* sTok = reinterpret_cast<int*>(sG + 128 * (p.ra + 4));                           // 3 x [128]

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t rank = kPair ? cluster_ctarank() : 0u;
  const int dt = blockIdx.x;                                   // 128 rows of dU
  // token blocks interleaved over the splits and walked from the END of the token range: all CTAs work in one window
  // that starts where k_tc_bwd_gz finished, i.e. on the part of g that is most likely still in L2 (c1 36.6 -> 35.8 us,
  // c3 164.8 -> 164.0 us against contiguous ranges walked forwards)
  const int n_mine = p.n_blocks > (int)blockIdx.y ? (p.n_blocks - 1 - (int)blockIdx.y) / (int)gridDim.y + 1 : 0;
  const int n_items = n_mine * p.n_src;
  const int tb0 = p.n_blocks - 1 - (int)blockIdx.y;
  constexpr int kBox = 64 * 128;                               // [64 tokens x 64 cols] bf16 = 8 KB
  const int nb_boxes = kPair ? p.r / 128 : p.r / 64;           // Zhat/gz boxes this CTA loads per item

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmG); tma_prefetch_desc(&tmZ); tma_prefetch_desc(&tmH); tma_prefetch_desc(&tmGz);
    tma_prefetch_desc(&tmDU);
    for (int s = 0; s < p.stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_init(acc_full, 1);
    fence_barrier_init();
  }
  if (warp == 1) {
    if (kPair) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(2u * (uint32_t)p.r) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(2u * (uint32_t)p.r) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  tc_fence_before_sync();
  if (kPair) cluster_sync_all(); else __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_d = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");

#ifdef MAPL_DBG
  const int dbg_cta = blockIdx.y * gridDim.x + blockIdx.x;
#define DU_DBG(i) { if (dbg_cta < 320) g_dbg[dbg_cta * 64 + (i)] = gtime(); }
#else
#define DU_DBG(i) {}
#endif
  if (threadIdx.x == 0) DU_DBG(0)
  if (warp >= 2 && p.tok != nullptr)
    scatter_gA(p, sG, sTok, blockIdx.y * gridDim.x + blockIdx.x, gridDim.x * gridDim.y);
  if (threadIdx.x == 64) DU_DBG(1)
  if (n_items > 0) {
    if (warp == 0) {
      if (elect_one()) {
        RingPos rp;
        int tb = tb0, src = 0;
        for (int it = 0; it < n_items; ++it, rp.next(p.stages)) {
          const int s = rp.st;
          mbar_wait(&empty[s], rp.ph ^ 1u);
          uint8_t* a = smem + (size_t)s * p.item_bytes;
          const CUtensorMap* ma = src ? &tmH : &tmG;
          const CUtensorMap* mb = src ? &tmGz : &tmZ;
          if (kPair) {
            if (rank == 0) mbar_arrive_expect_tx(&full[s], 2u * (uint32_t)p.item_bytes);
            tma_load_2d_pair(a, ma, &full[s], dt * 128, tb * 64, kEvictFirst);
            tma_load_2d_pair(a + kBox, ma, &full[s], dt * 128 + 64, tb * 64, kEvictFirst);
            for (int j = 0; j < nb_boxes; ++j)
              tma_load_2d_pair(a + 2 * kBox + j * kBox, mb, &full[s], (int)rank * (p.r / 2) + j * 64, tb * 64, kEvictLast);
          } else {
            mbar_arrive_expect_tx(&full[s], (uint32_t)p.item_bytes);
            tma_load_2d(a, ma, &full[s], dt * 128, tb * 64, kEvictFirst);
            tma_load_2d(a + kBox, ma, &full[s], dt * 128 + 64, tb * 64, kEvictFirst);
            for (int j = 0; j < nb_boxes; ++j) tma_load_2d(a + 2 * kBox + j * kBox, mb, &full[s], j * 64, tb * 64, kEvictLast);
          }
          if (++src == p.n_src) { src = 0; tb -= (int)gridDim.y; }
        }
      }
    } else if (warp == 1) {
      if (rank == 0 && elect_one()) {
        const uint32_t idesc = make_idesc_bf16(kPair ? 256 : 128, (uint32_t)p.r, true, true);
        const uint32_t smem0 = smem_u32(smem);
        RingPos rp;
        for (int it = 0; it < n_items; ++it, rp.next(p.stages)) {
          const int s = rp.st;
          mbar_wait(&full[s], rp.ph);
          if (it == 0) DU_DBG(2)
          if (it == n_items - 1) DU_DBG(3)
          tc_fence_after_sync();
          const uint32_t a = smem0 + (uint32_t)s * (uint32_t)p.item_bytes, b = a + 2 * kBox;
#pragma unroll
          for (int k = 0; k < 4; ++k) {     // 16 tokens (= 2 swizzle atoms of 8 rows) per UMMA
            const uint64_t da = desc_mnmajor_sw128(a + k * 2048, kBox), db = desc_mnmajor_sw128(b + k * 2048, kBox);
            // items alternate between two TMEM accumulators ([0,r) and [r,2r)), summed by the epilogue: the tensor core
            // adds into its accumulator with truncation, one-sided, so half the chain is half that bias of dU
            // (measured with one accumulator: -1.4e-4 relative at N = 2^20 tokens)
            const uint32_t acc = tmem_d + (uint32_t)(it & 1) * (uint32_t)p.r;
            if (kPair) umma_bf16_pair(acc, da, db, idesc, (it >= 2 || k != 0) ? 1u : 0u);
            else umma_bf16(acc, da, db, idesc, (it >= 2 || k != 0) ? 1u : 0u);
          }
          if (kPair) umma_commit_pair(&empty[s]); else umma_commit(&empty[s]);
        }
        if (kPair) umma_commit_pair(acc_full); else umma_commit(acc_full);
      }
    } else {
      // dU tile += accumulator: staged in the (now idle) ring as swizzled [128 rows x 32 floats] boxes and added by
      // TMA reductions -- whole 128-byte lines, where a row-per-thread red.global.add.v4 from the TMEM layout
      // sends 32 separate 16-byte reductions per instruction
      const int q = warp & 3, row = q * 32 + lane;
      mbar_wait(acc_full, 0);
      if (threadIdx.x == 64) DU_DBG(4)
      tc_fence_after_sync();
      for (int cc = 0; cc < p.r / 32; ++cc) {
        uint32_t v[32];
        tmem_ld32(tmem_d + ((uint32_t)(q * 32) << 16) + cc * 32, v);
        if (n_items >= 2) {            // the second accumulator (odd items)
          uint32_t w[32];
          tmem_ld32(tmem_d + ((uint32_t)(q * 32) << 16) + p.r + cc * 32, w);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) + __uint_as_float(w[i]));
        } else {
          tmem_ld_wait();
        }
#pragma unroll
        for (int i = 0; i < 8; ++i)
          *reinterpret_cast<float4*>(smem + (size_t)cc * kTileBytes + sw128_offset(row, i)) =
              make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]),
                          __uint_as_float(v[4 * i + 3]));
      }
      fence_proxy_async_smem();
      asm volatile("bar.sync 2, 128;" ::: "memory");
      if (threadIdx.x == 64) {
        for (int cc = 0; cc < p.r / 32; ++cc) tma_reduce_add_2d(&tmDU, smem + (size_t)cc * kTileBytes, cc * 32, dt * 128);
        tma_store_commit();
        tma_store_wait_all<0>();
      }
    }
  }
  if (threadIdx.x == 64) DU_DBG(5)
  tc_fence_before_sync();
  if (kPair) cluster_sync_all(); else __syncthreads();
  if (warp == 1) {
    tc_fence_after_sync();
    if (kPair) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"(2u * (uint32_t)p.r) : "memory");
    else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"(2u * (uint32_t)p.r) : "memory");
  }
}

}  // namespace
}  // namespace mapl
MAPL_DBG_READER(mapl_debug_read_bwd)
namespace mapl {

int tc_backward(const mapl_boundary_desc& d, const void* g, const void* H, const void* Z, const int32_t* codes,
                const float* codebooks, const int32_t* tok, const float* A, const TcPack& pk, void* gz_out,
                float* dU_out, float* dA_out, float* dB_out, void* dH_out, int accumulate, float* gA_ws,
                __nv_bfloat16* zhat_ws, cudaStream_t st) {
  if (!tc_shape_ok(d)) return MAPL_ERR_UNSUPPORTED;
  const int ra = tok ? d.anchor_rank : 0, kc = d.r + ra;

  MAPL_SMEM_OPT_IN(k_tc_bwd_gz, 227 * 1024);
  MAPL_SMEM_OPT_IN(k_tc_bwd_du<true>, 227 * 1024);
  MAPL_SMEM_OPT_IN(k_tc_bwd_du<false>, 227 * 1024);
  const uint64_t N = (uint64_t)d.n_tokens, dd = (uint64_t)d.d, rr = (uint64_t)d.r;

  // zhat operand for dU
  const void* zhat = Z;
  if (codes) zhat = zhat_ws;        // written by k_tc_bwd_gz (dequantisation fused under its g stream)

  {  // ---- gz, gA, dH (+ zero fill of the overwrite outputs)
    BwdGzParams p;
    p.gA = gA_ws; p.gz_out = reinterpret_cast<__nv_bfloat16*>(gz_out);
    p.z0 = p.z1 = p.z2 = nullptr; p.n0 = p.n1 = p.n2 = 0;
    if (!accumulate) {
      p.z0 = dU_out; p.n0 = (long long)d.d * d.r;
      if (ra) { p.z1 = dA_out; p.n1 = (long long)d.vocab * ra; }
      if (ra && dB_out) { p.z2 = dB_out; p.n2 = (long long)ra * d.d; }
    }
    p.nq = tc_pairs_per_cluster();
    p.N = d.n_tokens; p.d = d.d; p.r = d.r; p.ra = ra; p.tile_m = p.nq == 2 ? tc_tile_m4(d.n_tokens) : tc_tile_m(d.n_tokens);
    p.do_dh = dH_out ? 1 : 0;
    p.stage1_bytes = kTileBytes + kc * 64;
    const size_t budget = 227 * 1024 - (size_t)kOutBufs * kTileBytes - 1024 - 1024;   // region R
    p.stages1 = (int)(budget / p.stage1_bytes);
    if (p.stages1 > 8) p.stages1 = 8;
    if (p.stages1 > d.d / 64) p.stages1 = d.d / 64;
    if (p.stages1 < 2) return MAPL_ERR_UNSUPPORTED;
    p.b_stages = (int)((budget - (size_t)(d.r / 64) * kTileBytes) / kTileBytes);
    if (p.b_stages > 16) p.b_stages = 16;
    if (p.b_stages < 2) return MAPL_ERR_UNSUPPORTED;
    const size_t ring1 = (size_t)p.stages1 * p.stage1_bytes,
                 ring2 = (size_t)(d.r / 64) * kTileBytes + (size_t)p.b_stages * kTileBytes;
    const size_t smem = (ring1 > ring2 ? ring1 : ring2) + (size_t)kOutBufs * kTileBytes + 1024 + 1024;
    static_assert(kOutBufs == 4, "gA staging: ra / 32 pieces over four boxes");
    p.ga_tma = (ra == 64 || ra == 128) ? 1 : 0;
    p.codes = codes; p.codebooks = codebooks; p.zhat_out = zhat_ws; p.L = d.rvq_levels; p.K = d.rvq_k;
    CUtensorMap tmG, tmWu, tmWb, tmWd, tmO, tmGz, tmGA;
    if (!make_tmap_bf16_2d(&tmGz, gz_out, N, rr, rr, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
    // gA map: unused unless ga_tma, but must be valid
    if (p.ga_tma) { if (!make_tmap_f32_2d(&tmGA, gA_ws, N, (uint64_t)ra, (uint64_t)ra, 32, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA; }
    else tmGA = tmGz;
    // dH map: when dH is skipped the map is unused but must be valid
    if (!make_tmap_bf16_2d(&tmO, dH_out ? dH_out : g, N, dd, dd, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmG, g, N, dd, dd, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmWu, pk.WB, (uint64_t)pk.kc, dd, dd, 64, (uint32_t)(d.r / 2 / p.nq))) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmWb, pk.WB, (uint64_t)pk.kc, dd, dd, 64, (uint32_t)((ra ? ra : 64) / 2 / p.nq))) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmWd, pk.Wd, dd, (uint64_t)pk.kc, (uint64_t)pk.kc, 64, (uint32_t)(kChunkN / 2 / p.nq))) return MAPL_ERR_CUDA;
    const unsigned cl = 2u * (unsigned)p.nq;
    const unsigned tiles = ((unsigned)((d.n_tokens + p.tile_m - 1) / p.tile_m) + cl - 1u) / cl * cl;   // whole clusters
    KernelScope ks(KID_TC_BWD_GZ, st);
    MAPL_CUDA_CHECK(launch_pdl_cluster(k_tc_bwd_gz, dim3(tiles), dim3(kThreads), smem, st, cl, tmG, tmWu, tmWb, tmWd, tmO, tmGz, tmGA, p));
  }
  {  // ---- dU (+ dA scatter)
    BwdDuParams p;
    p.dU = dU_out; p.N = d.n_tokens; p.d = d.d; p.r = d.r; p.n_src = H ? 2 : 1;
    p.tok = ra ? tok : nullptr; p.gA = gA_ws; p.dA = dA_out; p.ra = ra;
    const int n_dt = d.d / 128;
    const bool pair = d.r >= 128 && n_dt % 2 == 0;
    p.item_bytes = 2 * 64 * 128 + (pair ? d.r / 128 : d.r / 64) * 64 * 128;      // per CTA
    const size_t scatter_bytes = ra ? (size_t)128 * (ra + 4) * 4 + 3 * 512 : 0;
    p.stages = (int)((227 * 1024 - 2048 - scatter_bytes) / p.item_bytes);
    if (p.stages > 8) p.stages = 8;
    if (p.stages < 2 || (size_t)p.stages * p.item_bytes < (size_t)(d.r / 32) * kTileBytes) return MAPL_ERR_UNSUPPORTED;   // ring doubles as the dU staging
    p.n_blocks = (int)((d.n_tokens + 63) / 64);
    int S = 148 / n_dt;
    if (S < 1) S = 1;
    if (S > p.n_blocks) S = p.n_blocks;
    p.blocks_per_split = (p.n_blocks + S - 1) / S;
    S = (p.n_blocks + p.blocks_per_split - 1) / p.blocks_per_split;
    const size_t smem = (size_t)p.stages * p.item_bytes + 1024 + 512 + scatter_bytes;
    CUtensorMap tmG, tmZ, tmH, tmGz, tmDU;
    if (!make_tmap_f32_2d(&tmDU, dU_out, dd, rr, rr, 32, 128)) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmG, g, N, dd, dd, 64, 64)) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmZ, zhat, N, rr, rr, 64, 64)) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmH, H ? H : g, N, dd, dd, 64, 64)) return MAPL_ERR_CUDA;
    if (!make_tmap_bf16_2d(&tmGz, gz_out, N, rr, rr, 64, 64)) return MAPL_ERR_CUDA;
    KernelScope ks(KID_TC_BWD_DU, st);
    if (pair) MAPL_CUDA_CHECK(launch_pdl_pair(k_tc_bwd_du<true>, dim3(n_dt, S), dim3(kThreadsDu), smem, st, tmG, tmZ, tmH, tmGz, tmDU, p));
    else MAPL_CUDA_CHECK(launch_pdl(k_tc_bwd_du<false>, dim3(n_dt, S), dim3(kThreadsDu), smem, st, tmG, tmZ, tmH, tmGz, tmDU, p));
  }
  if (dB_out && ra) {   // dB += A[tok]^T g  (P_p is frozen in the paper: optional, fp32 SIMT)
    GemmArgs ga;
    ga.M = ra; ga.N = d.d; ga.K[0] = (int)d.n_tokens;
    ga.A[0].p = A; ga.A[0].so = 1; ga.A[0].sk = ra; ga.A[0].gather = tok; ga.A[0].gmode = 2;
    ga.B[0].p = g; ga.B[0].bf16 = 1; ga.B[0].so = 1; ga.B[0].sk = d.d;
    ga.C = dB_out; ga.ldc = d.d; ga.atomic = 1; ga.splits = (int)((d.n_tokens + 1023) / 1024);
    MAPL_RETURN_IF(simt_gemm(ga, st));
  }
  return MAPL_OK;
}

}  // namespace mapl
