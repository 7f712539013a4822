// tc_decode.cu -- mapl_decode on the tensor cores:  Hhat = [Zhat | A[tok]] . [U | B^T]^T
// (Eq. 2 with the factorised anchor of PAPER.md:106 Eq. 3 folded in as extra K columns).
//
// One CTA per token tile (tile_m <= 128 tokens, sized so the grid fills the 148 SMs evenly).
//   A operand  [128 x Kc] bf16, K-major SW128, resident for the CTA's lifetime:
//                columns [0,r): Zhat -- TMA from the wire payload, or dequantised from the RVQ
//                codes by the epilogue warps (gather-sum of codewords, fp32, rounded once);
//                columns [r,Kc): rows A[tok] gathered from the fp32 table by the epilogue warps.
//   B operand  Wd pack [d, Kc] bf16 streamed in [128 x 64] tiles through a TMA/mbarrier ring.
//   D, epilogue: see tc_tile_ops.cuh.
// Roofline: HBM (writes d*2 B/token).
#include "profile.cuh"
#include "tc_codec.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

constexpr int kThreads = 192;

struct DecodeParams {
  const int32_t* codes; const float* codebooks;   // RVQ dequant (codes != nullptr)
  const int32_t* tok; const float* A;             // anchor gather (tok != nullptr)
  long long N;
  int d, r, ra, L, K;
  int tile_m, b_stages, z_from_tma;
};

__global__ void __launch_bounds__(kThreads, 1)
k_tc_decode(const __grid_constant__ CUtensorMap tmZ, const __grid_constant__ CUtensorMap tmW,
            const __grid_constant__ CUtensorMap tmO, const DecodeParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  ChunkPipe c;
  c.nkb = (p.r + p.ra) / 64; c.nchunks = p.d / kChunkN; c.b_stages = p.b_stages;
  c.sA = smem;
  c.sOut = c.sA + (size_t)c.nkb * kTileBytes;
  c.sB = c.sOut + (size_t)kOutBufs * kTileBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(c.sB + (size_t)p.b_stages * kTileBytes);
  c.b_full = bars; c.b_empty = c.b_full + p.b_stages;
  c.acc_full = c.b_empty + p.b_stages; c.acc_empty = c.acc_full + kAccStages;
  uint64_t* a_full = c.acc_empty + kAccStages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(a_full + 1);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const long long m0 = (long long)blockIdx.x * p.tile_m;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmZ); tma_prefetch_desc(&tmW); tma_prefetch_desc(&tmO);
    chunk_init_barriers(c);
    mbar_init(a_full, 1 + 4);                 // producer (expect_tx) + one arrive per epilogue warp
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<512>(tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  c.tmem_base = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");       // everything below touches global memory

  if (warp == 0) {
    if (elect_one()) {
      if (p.z_from_tma) {
        mbar_arrive_expect_tx(a_full, (uint32_t)((p.r / 64) * p.tile_m * 128));
        for (int kb = 0; kb < p.r / 64; ++kb)
          tma_load_2d(c.sA + (size_t)kb * kTileBytes, &tmZ, a_full, kb * 64, (int)m0, kEvictFirst);
      } else {
        mbar_arrive(a_full);
      }
      chunk_produce(c, &tmW);
    }
  } else if (warp == 1) {
    if (elect_one()) {
      mbar_wait(a_full, 0);
      tc_fence_after_sync();
      chunk_mma(c);
    }
  } else {
    const int q = warp & 3;
    const int row = q * 32 + lane;                      // token row inside the tile == TMEM lane
    const long long m = m0 + row;
    const bool live = row < p.tile_m && m < p.N;
    // ---- A operand columns produced by threads: dequantised zhat and gathered anchor rows
    if (!p.z_from_tma) {
      const float* rowp[8];
#pragma unroll
      for (int l = 0; l < 8; ++l)
        rowp[l] = p.codebooks + ((long long)(l < p.L ? l : 0) * p.K + ((live && l < p.L) ? __ldg(p.codes + m * p.L + l) : 0)) * p.r;
      for (int cc = 0; cc < p.r / 8; ++cc) {            // 8 columns = one 16-byte chunk
        float s[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (live) {
#pragma unroll
          for (int l = 0; l < 8; ++l) {
            if (l >= p.L) break;
            const float4* src = reinterpret_cast<const float4*>(rowp[l] + cc * 8);
            const float4 x = __ldg(src), y = __ldg(src + 1);
            s[0] += x.x; s[1] += x.y; s[2] += x.z; s[3] += x.w; s[4] += y.x; s[5] += y.y; s[6] += y.z; s[7] += y.w;
          }
        }
        const uint4 o = make_uint4(pack_bf16x2(s[0], s[1]), pack_bf16x2(s[2], s[3]), pack_bf16x2(s[4], s[5]), pack_bf16x2(s[6], s[7]));
        *reinterpret_cast<uint4*>(c.sA + (size_t)(cc / 8) * kTileBytes + sw128_offset(row, cc % 8)) = o;
      }
    }
    if (p.ra > 0) {
      const long long t = live ? (long long)__ldg(p.tok + m) : 0;
      const float4* src = reinterpret_cast<const float4*>(p.A + t * p.ra);
      for (int c0 = 0; c0 < p.ra / 8; c0 += 4) {       // 8 independent 16-byte loads in flight per thread
        float4 x[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = live ? __ldg(src + c0 * 2 + i) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int cc = c0 + i;
          const uint4 o = make_uint4(pack_bf16x2(x[2 * i].x, x[2 * i].y), pack_bf16x2(x[2 * i].z, x[2 * i].w),
                                     pack_bf16x2(x[2 * i + 1].x, x[2 * i + 1].y), pack_bf16x2(x[2 * i + 1].z, x[2 * i + 1].w));
          *reinterpret_cast<uint4*>(c.sA + (size_t)(p.r / 64 + cc / 8) * kTileBytes + sw128_offset(row, cc % 8)) = o;
        }
      }
    }
    fence_proxy_async_smem();
    __syncwarp();
    if (lane == 0) mbar_arrive(a_full);
    chunk_epilogue(c, &tmO, (int)m0);
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc<512>(c.tmem_base);
  }
}

}  // namespace

int tc_decode(const mapl_boundary_desc& d, const void* Z, const int32_t* codes, const float* codebooks,
              const int32_t* tok, const float* A, const TcPack& pk, void* Hhat_out, cudaStream_t st) {
  if (!tc_shape_ok(d)) return MAPL_ERR_UNSUPPORTED;
  const int ra = d.anchor_rank, kc = d.r + ra, nkb = kc / 64;
  DecodeParams p;
  p.codes = codes; p.codebooks = codebooks; p.tok = ra ? tok : nullptr; p.A = A;
  p.N = d.n_tokens; p.d = d.d; p.r = d.r; p.ra = ra; p.L = d.rvq_levels; p.K = d.rvq_k;
  p.tile_m = tc_tile_m(d.n_tokens);
  p.z_from_tma = codes ? 0 : 1;
  const size_t fixed = (size_t)(nkb + kOutBufs) * kTileBytes + 1024 + 512;
  p.b_stages = (int)((227 * 1024 - fixed) / kTileBytes);
  if (p.b_stages > 8) p.b_stages = 8;
  if (p.b_stages < 2) return MAPL_ERR_UNSUPPORTED;
  const size_t smem = fixed + (size_t)p.b_stages * kTileBytes;
  CUtensorMap tmZ, tmW, tmO;
  // Z: [N, r]; when zhat comes from codes the map is unused but must be valid: point it at the pack
  const void* zbase = codes ? (const void*)pk.Wd : Z;
  if (!make_tmap_bf16_2d(&tmZ, zbase, codes ? (uint64_t)d.d : (uint64_t)d.n_tokens, codes ? (uint64_t)kc : (uint64_t)d.r,
                         codes ? (uint64_t)kc : (uint64_t)d.r, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmW, pk.Wd, (uint64_t)d.d, (uint64_t)kc, (uint64_t)kc, 64, kChunkN)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmO, Hhat_out, (uint64_t)d.n_tokens, (uint64_t)d.d, (uint64_t)d.d, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
  static bool attr_done = false;
  if (!attr_done) {
    MAPL_CUDA_CHECK(cudaFuncSetAttribute(k_tc_decode, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    attr_done = true;
  }
  const unsigned tiles = (unsigned)((d.n_tokens + p.tile_m - 1) / p.tile_m);
  KernelScope ks(KID_TC_DECODE, st);
  MAPL_CUDA_CHECK(launch_pdl(k_tc_decode, dim3(tiles), dim3(kThreads), smem, st, tmZ, tmW, tmO, p));
  return MAPL_OK;
}

}  // namespace mapl
