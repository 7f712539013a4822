// tc_encode_rvq.cu -- mapl_encode with residual VQ on the tensor cores: projection and all RVQ
// levels in ONE kernel, z never leaves the chip (Eq. 1; Sec. 3.5;
// readings S3-S5 of DESIGN.md).
//
// One CTA per token tile (<= 128 tokens; one TMEM lane = one token); CTAs work in pairs (cluster of 2,
// cta_group::2 MMAs of M = 256): each CTA loads half of every parameter / codebook tile.
//   phase 1   z = H (U_hi + U_lo)      H tiles by TMA (HBM, evict-first), the two bf16 split terms
//             of U^T from the L2-resident pack; fp32 accumulator [128 x r] in TMEM columns [0,r).
//             bf16 H is exact and U_hi + U_lo carries 16 mantissa bits, so z is fp32-accurate.
//   level l   rho (fp32) stays in TMEM columns [0,r); its fp16 rounding, scaled per token by a power
//             of two so that max|rho_j| lies in [0.5,1), is the resident A operand (the codebook
//             copy is fp16 too, scaled per level: 11 significant bits instead of bf16's 8).
//             Codebook tiles [128 codewords x 64] stream through a TMA ring; per 128-codeword
//             chunk one accumulator stage S = rho_f16 . C_f16^T  (2 stages, TMEM cols 256..511).
//             Epilogue (thread = token): coarse score s_k = 0.5||c_k||^2 - S_k, running minimum,
//             and every k with  s_k <= running min + margin  is recorded as a candidate, where
//               margin = 2 E,   E = 2^-10 * 1.05 * ||rho|| * max_k ||c_k||  >=  |s_coarse - s_exact|
//             (fp16 rounding of both operands, Cauchy-Schwarz).  The true minimiser is therefore
//             always among the candidates; they are re-scored in exact fp32 (rho from TMEM, the
//             fp32 codeword from L2), lowest index winning ties (S4).  Then rho -= C[l, k*].
//             A thread's candidate list holds kNE 32-codeword pieces; when it is full it keeps the
//             pieces with the lowest minima, and only a left-out piece whose minimum is within the
//             FINAL threshold (the threshold only tightens during the scan) sends the warp to the
//             exhaustive fp32 pass over all K codewords (duplicate-heavy codebooks).
// Roofline: tensor at config 3 (K r = 1M per level), HBM/ALU at config 2.
#include <float.h>

#include "profile.cuh"
#include "tc_codec.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

// scan / re-score threads per token (warps per TMEM lane quarter): 2 or 4.  Measured: 4 (16 scan warps, 96 registers)
// is SLOWER -- c2 encode 59.7 -> 62.2 us, c3 239 -> 271 us: the per-warp cost of a chunk (TMEM load, wait, barrier
// arrive, list bookkeeping) does not shrink with the piece count and the 512-thread exchanges cost more.
#ifndef MAPL_RVQ_PARTS
#define MAPL_RVQ_PARTS 2
#endif
constexpr int kParts = MAPL_RVQ_PARTS;
constexpr int kEpi = 128 * kParts;       // epilogue threads
constexpr int kThreads = 64 + kEpi;      // warp 0 TMA, warp 1 MMA, then kParts x 4 scan / re-score warps
constexpr int kChunk = 128;        // codewords per accumulator stage (UMMA N)
constexpr int kAccCol0 = 256;      // TMEM column of score stage 0
constexpr int kNE = 8;             // candidate-list entries per thread (one entry = one 32-codeword piece)

struct RvqParams {
  const float* C;        // [L,K,r] fp32 codebooks (exact re-scoring, residual update)
  const float* hn;       // [L*K] 0.5 ||c||^2
  const float* cmax;     // [L] max_k ||c_k||
  const float* cscale;   // [8+l] = 2^e_l: the fp16 codebook copy is C * 2^-e_l
  const int32_t* tok; const float* Tc;   // optional sender-side centring (Eq. 1): z -= Tc[tok], Tc [V,r] fp32
  __nv_bfloat16* Zq;     // optional [N,r]
  int32_t* codes;        // [N,L]
  long long N;
  int d, r, L, K, tile_m;
  int stages1, stage1_bytes, ring_tiles;
};

// smem carve-up (after 1024-byte alignment):
//   region R  = max(phase-1 ring, rho operand tiles + codebook ring)
//   sHn [K] fp32 | candidate lists [kNE][kEpi] x (m32, piece, mask) | exchange [5][kParts][128] | barriers | tmem slot
struct Smem {
  uint8_t* ring1; uint8_t* sRho; uint8_t* ringC;
  float* sHn; float* eM; int* eP; uint32_t* eMask;
  float* xch;            // [5][kParts][128]: per (part, token) best / score / k / n2 / amax exchanged by the warps of a quarter
  uint64_t* s1_full; uint64_t* s1_empty; uint64_t* z_full;
  uint64_t* c_full; uint64_t* c_empty; uint64_t* acc_full; uint64_t* acc_empty; uint64_t* rho_ready;
  uint32_t* tmem_slot;
};

__host__ __device__ inline size_t rvq_regionR(const RvqParams& p) {
  const size_t ring1 = (size_t)p.stages1 * p.stage1_bytes;
  const size_t lvl = (size_t)(p.r / 64) * kTileBytes + (size_t)p.ring_tiles * kHalfTileBytes;
  return ring1 > lvl ? ring1 : lvl;
}
__host__ __device__ inline size_t rvq_tail_bytes(const RvqParams& p) {
  return (size_t)p.K * 4 + (size_t)kNE * kEpi * 12 + 5 * kEpi * 4 + 1024;
}

__device__ __forceinline__ Smem carve_smem(uint8_t* base, const RvqParams& p) {
  Smem s;
  s.ring1 = base;
  s.sRho = base;
  s.ringC = base + (size_t)(p.r / 64) * kTileBytes;
  uint8_t* t = base + rvq_regionR(p);
  s.sHn = reinterpret_cast<float*>(t); t += (size_t)p.K * 4;
  s.eM = reinterpret_cast<float*>(t); t += kNE * kEpi * 4;
  s.eP = reinterpret_cast<int*>(t); t += kNE * kEpi * 4;
  s.eMask = reinterpret_cast<uint32_t*>(t); t += kNE * kEpi * 4;
  s.xch = reinterpret_cast<float*>(t); t += 5 * kEpi * 4;
  uint64_t* b = reinterpret_cast<uint64_t*>(t);
  s.s1_full = b; b += p.stages1;
  s.s1_empty = b; b += p.stages1;
  s.z_full = b; b += 1;
  s.c_full = b; b += p.ring_tiles;
  s.c_empty = b; b += p.ring_tiles;
  s.acc_full = b; b += 2;
  s.acc_empty = b; b += 2;
  s.rho_ready = b; b += 1;
  s.tmem_slot = reinterpret_cast<uint32_t*>(b);
  return s;
}

// exact fp32 score of codeword row `crow` against this thread's residual (TMEM columns [0,r)):
// 0.5||c||^2 - rho.c.  Warp-convergent (tcgen05.ld is .sync.aligned); lanes without work pass any
// valid row and ignore the result.
__device__ __forceinline__ float exact_score(uint32_t tmem_row, const float* __restrict__ crow, float hn, int r) {
  // the row loads (L2 latency) of TWO 32-column pieces are in flight together (r is a multiple of 64); the residual
  // pieces are read from TMEM one at a time to keep the register count down
  float dot = 0.f;
  for (int pc = 0; pc < r / 32; pc += 2) {
    const float4* c4 = reinterpret_cast<const float4*>(crow + pc * 32);
    float4 c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = __ldg(c4 + i);
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      uint32_t v[32];
      tmem_ld32(tmem_row + (pc + u) * 32, v);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        dot = fmaf(__uint_as_float(v[4 * i + 0]), c[8 * u + i].x, dot);
        dot = fmaf(__uint_as_float(v[4 * i + 1]), c[8 * u + i].y, dot);
        dot = fmaf(__uint_as_float(v[4 * i + 2]), c[8 * u + i].z, dot);
        dot = fmaf(__uint_as_float(v[4 * i + 3]), c[8 * u + i].w, dot);
      }
    }
  }
  return hn - dot;
}

// The kParts warps of a TMEM lane quarter split the residual by 32-column pieces: part h owns the
// pieces pc with pc % kParts == h.
// Step 1 of a residual update: rho <- rho - sub on the own pieces (sub == nullptr: rho unchanged);
// returns the partial ||rho||^2 and max|rho_j| of those pieces.  Warp-convergent.
__device__ __forceinline__ void rho_subtract(uint32_t tmem_row, const float* __restrict__ sub, int r, int h, float* n2_out,
                                             float* amax_out) {
  float n2 = 0.f, amax = 0.f;
  for (int pc = h; pc < r / 32; pc += kParts) {
    uint32_t v[32];
    tmem_ld32(tmem_row + pc * 32, v);
    tmem_ld_wait();
    if (sub != nullptr) {
      const float4* c4 = reinterpret_cast<const float4*>(sub + pc * 32);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float4 c = __ldg(c4 + i);
        v[4 * i + 0] = __float_as_uint(__uint_as_float(v[4 * i + 0]) - c.x);
        v[4 * i + 1] = __float_as_uint(__uint_as_float(v[4 * i + 1]) - c.y);
        v[4 * i + 2] = __float_as_uint(__uint_as_float(v[4 * i + 2]) - c.z);
        v[4 * i + 3] = __float_as_uint(__uint_as_float(v[4 * i + 3]) - c.w);
      }
      tmem_st32(tmem_row + pc * 32, v);
    }
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const float x = __uint_as_float(v[i]);
      n2 = fmaf(x, x, n2);
      amax = fmaxf(amax, fabsf(x));
    }
  }
  if (sub != nullptr) tmem_st_wait();
  *n2_out = n2; *amax_out = amax;
}

// Step 2: fp16(rho * 2^-e) of the own pieces into the swizzled A-operand tiles, 2^-e chosen from the
// row's max|rho_j| so that it lands in [0.5,1); returns 2^e.  Warp-convergent.
__device__ __forceinline__ float rho_to_operand(uint32_t tmem_row, uint8_t* sRho, int row, int r, int h, float amax) {
  int eb = (int)((__float_as_uint(amax) >> 23) & 0xffu);
  eb = eb < 2 ? 126 : (eb > 250 ? 250 : eb);
  const float inv = __uint_as_float((uint32_t)(253 - eb) << 23);
  for (int pc = h; pc < r / 32; pc += kParts) {
    uint32_t v[32];
    tmem_ld32(tmem_row + pc * 32, v);
    tmem_ld_wait();
    uint8_t* tile = sRho + (size_t)(pc / 2) * kTileBytes;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      uint4 o;
      o.x = pack_f16x2(__uint_as_float(v[8 * i + 0]) * inv, __uint_as_float(v[8 * i + 1]) * inv);
      o.y = pack_f16x2(__uint_as_float(v[8 * i + 2]) * inv, __uint_as_float(v[8 * i + 3]) * inv);
      o.z = pack_f16x2(__uint_as_float(v[8 * i + 4]) * inv, __uint_as_float(v[8 * i + 5]) * inv);
      o.w = pack_f16x2(__uint_as_float(v[8 * i + 6]) * inv, __uint_as_float(v[8 * i + 7]) * inv);
      *reinterpret_cast<uint4*>(tile + sw128_offset(row, (pc & 1) * 4 + i)) = o;
    }
  }
  return __uint_as_float((uint32_t)(eb + 1) << 23);
}

// named barrier 1 over the epilogue warps
__device__ __forceinline__ void epi_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kEpi) : "memory"); }

__global__ void __launch_bounds__(kThreads, 1)
k_tc_encode_rvq(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmWhi,
                const __grid_constant__ CUtensorMap tmWlo, const __grid_constant__ CUtensorMap tmC,
                const RvqParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const Smem s = carve_smem(smem, p);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t rank = cluster_ctarank();
  const long long m0 = (long long)blockIdx.x * p.tile_m;
  const int nkb1 = p.d / 64, nkb = p.r / 64, nchunks = p.K / kChunk;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmH); tma_prefetch_desc(&tmWhi); tma_prefetch_desc(&tmWlo); tma_prefetch_desc(&tmC);
    for (int i = 0; i < p.stages1; ++i) { mbar_init(&s.s1_full[i], 1); mbar_init(&s.s1_empty[i], 1); }
    mbar_init(s.z_full, 1);
    for (int i = 0; i < p.ring_tiles; ++i) { mbar_init(&s.c_full[i], 1); mbar_init(&s.c_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s.acc_full[i], 1); mbar_init(&s.acc_empty[i], 8 * kParts); }
    mbar_init(s.rho_ready, 8 * kParts);               // leader's barriers collect the epilogue warps of both CTAs
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(s.tmem_slot);
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem_base = *s.tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");       // everything below touches global memory
  if (warp == 0) { DBG(0) }

  if (warp == 0) {
    // ------------------------------------------------------------ TMA producer
    if (elect_one()) {
      const uint32_t w_tile = (uint32_t)p.r * 64;          // this CTA's half (r/2 rows) of a U^T tile
      for (int kb = 0; kb < nkb1; ++kb) {
        const int st = kb % p.stages1;
        mbar_wait(&s.s1_empty[st], ((kb / p.stages1) & 1) ^ 1);
        if (rank == 0) mbar_arrive_expect_tx(&s.s1_full[st], 2u * ((uint32_t)(p.tile_m * 128) + 2 * w_tile));
        uint8_t* a = s.ring1 + (size_t)st * p.stage1_bytes;
        tma_load_2d_pair(a, &tmH, &s.s1_full[st], kb * 64, (int)m0, kEvictFirst);
        tma_load_2d_pair(a + kTileBytes, &tmWhi, &s.s1_full[st], kb * 64, (int)rank * (p.r / 2), kEvictLast);
        tma_load_2d_pair(a + kTileBytes + w_tile, &tmWlo, &s.s1_full[st], kb * 64, (int)rank * (p.r / 2), kEvictLast);
      }
      mbar_wait(s.z_full, 0);             // phase-1 MMAs have consumed region R: it may be reused
      int it = 0;
      for (int l = 0; l < p.L; ++l)
        for (int c = 0; c < nchunks; ++c)
          for (int kb = 0; kb < nkb; ++kb, ++it) {
            const int st = it % p.ring_tiles;
            mbar_wait(&s.c_empty[st], ((it / p.ring_tiles) & 1) ^ 1);
            if (rank == 0) mbar_arrive_expect_tx(&s.c_full[st], 2 * kHalfTileBytes);
            tma_load_2d_pair(s.ringC + (size_t)st * kHalfTileBytes, &tmC, &s.c_full[st], kb * 64,
                             l * p.K + c * kChunk + (int)rank * (kChunk / 2), kEvictLast);
          }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer
    if (rank == 0 && elect_one()) {
      const uint32_t idesc1 = make_idesc_bf16(256, (uint32_t)p.r, false, false);
      for (int kb = 0; kb < nkb1; ++kb) {
        const int st = kb % p.stages1;
        mbar_wait(&s.s1_full[st], (kb / p.stages1) & 1);
        tc_fence_after_sync();
        const uint32_t a = smem_u32(s.ring1 + (size_t)st * p.stage1_bytes);
        const uint32_t bh = a + kTileBytes, bl = bh + p.r * 64;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint64_t da = desc_kmajor_sw128(a + k * 32);
          // even / odd k-blocks accumulate into two TMEM regions ([0,r) and the still unused score stages at
          // [256,256+r)): the tensor core truncates when it adds into its accumulator, and halving the chain of
          // MMAs halves that one-sided error of z (tc_stiefel.cu measures it); the epilogue adds the two halves
          const uint32_t acc = tmem_base + (uint32_t)(kb & 1) * kAccCol0;
          umma_bf16_pair(acc, da, desc_kmajor_sw128(bh + k * 32), idesc1, (kb >= 2) || k != 0);
          umma_bf16_pair(acc, da, desc_kmajor_sw128(bl + k * 32), idesc1, 1);
        }
        umma_commit_pair(&s.s1_empty[st]);
      }
      umma_commit_pair(s.z_full);
      const uint32_t idesc2 = make_idesc_f16(256, kChunk);
      int it = 0, cg = 0;
      for (int l = 0; l < p.L; ++l) {
        mbar_wait_cluster(s.rho_ready, l & 1);    // fp16 residuals of level l are in sRho of both CTAs
        tc_fence_after_sync();
        for (int c = 0; c < nchunks; ++c, ++cg) {
          const int as = cg & 1;
          mbar_wait_cluster(&s.acc_empty[as], ((cg >> 1) & 1) ^ 1);
          if (cg < 8) DBGT(24 + cg)
          tc_fence_after_sync();
          const uint32_t tmem_d = tmem_base + kAccCol0 + as * kChunk;
          for (int kb = 0; kb < nkb; ++kb, ++it) {
            const int st = it % p.ring_tiles;
            mbar_wait(&s.c_full[st], (it / p.ring_tiles) & 1);
            tc_fence_after_sync();
            const uint32_t a = smem_u32(s.sRho + (size_t)kb * kTileBytes), b = smem_u32(s.ringC + (size_t)st * kHalfTileBytes);
#pragma unroll
            for (int k = 0; k < 4; ++k)
              umma_bf16_pair(tmem_d, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(b + k * 32), idesc2, (kb | k) != 0);
            umma_commit_pair(&s.c_empty[st]);
          }
          umma_commit_pair(&s.acc_full[as]);
          if (cg < 8) DBGT(32 + cg)
        }
      }
    }
  } else {
    // ------------------------------------------------------------ epilogue: 4 kParts warps, kParts threads per token
    // q = TMEM lane quarter, h = which part of the 32-codeword pieces / 32-column pieces this warp owns
    const int q = warp & 3, h = (warp - 2) >> 2, row = q * 32 + lane, et = threadIdx.x - 64;
    const long long m = m0 + row;
    const bool live = row < p.tile_m && m < p.N;
    const uint32_t tmem_row = tmem_base + ((uint32_t)(q * 32) << 16);
    const unsigned full = 0xffffffffu;
    float* xBest = s.xch; float* xScore = s.xch + kEpi; int* xK = reinterpret_cast<int*>(s.xch + 2 * kEpi);
    float* xN2 = s.xch + 3 * kEpi; float* xAmax = s.xch + 4 * kEpi;
    const int mine = h * 128 + row;
    float* eM = s.eM + mine; int* eP = s.eP + mine; uint32_t* eMask = s.eMask + mine;   // entry e at [e * kEpi]
    int code_l[8];
#pragma unroll
    for (int l = 0; l < 8; ++l) code_l[l] = 0;
    const uint32_t sHn_u32 = smem_u32(s.sHn);

    mbar_wait(s.z_full, 0);
    if (warp == 2) { DBG(1) }
    tc_fence_after_sync();
    float n2, amax;
    if (nkb1 >= 2) {                     // z = even-k-block half + odd-k-block half (see the MMA issuer)
      for (int pc = h; pc < p.r / 32; pc += kParts) {
        uint32_t v[32], w[32];
        tmem_ld32(tmem_row + pc * 32, v);
        tmem_ld32(tmem_row + kAccCol0 + pc * 32, w);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) + __uint_as_float(w[i]));
        tmem_st32(tmem_row + pc * 32, v);
      }
      tmem_st_wait();
    }
    // centring: the first residual is z - Tc[tok] (dead rows subtract row 0: any valid row keeps the warp convergent)
    const float* csub = p.Tc != nullptr ? p.Tc + (live ? (long long)__ldg(p.tok + m) * p.r : 0) : nullptr;
    rho_subtract(tmem_row, csub, p.r, h, &n2, &amax);
    xN2[mine] = n2; xAmax[mine] = amax;
    epi_sync();
    n2 = 0.f; amax = 0.f;
#pragma unroll
    for (int hh = 0; hh < kParts; ++hh) { n2 += xN2[hh * 128 + row]; amax = fmaxf(amax, xAmax[hh * 128 + row]); }
    float unscale = rho_to_operand(tmem_row, s.sRho, row, p.r, h, amax);
    fence_proxy_async_smem();
    tc_fence_before_sync();
    __syncwarp();
    if (lane == 0) mbar_arrive_leader(s.rho_ready);

    int cg = 0;
#pragma unroll 1
    for (int l = 0; l < p.L; ++l) {
      const float* Cl = p.C + (long long)l * p.K * p.r;
      for (int i = et; i < p.K / 4; i += kEpi)
        reinterpret_cast<float4*>(s.sHn)[i] = __ldg(reinterpret_cast<const float4*>(p.hn + (long long)l * p.K) + i);
      epi_sync();
      if (warp == 2 && l < 4) { DBG(4 + l * 4) }
      const float margin = 0.001953125f * 1.05f * sqrtf(n2) * __ldg(p.cmax + l);
      const float nsc = -unscale * __ldg(p.cscale + 8 + l);     // coarse S -> rho.c

      float best = FLT_MAX;
      int cnt = 0;
      float dropped = FLT_MAX;           // lowest piece minimum that found no room in the list
      for (int c = 0; c < nchunks; ++c, ++cg) {
        const int as = cg & 1;
        mbar_wait(&s.acc_full[as], (cg >> 1) & 1);
        if (threadIdx.x == 64 && cg < 8) DBGT(40 + cg)
        tc_fence_after_sync();
        uint32_t v[4 / kParts][32];            // this warp's pieces of the chunk: h, h + kParts, ...
#pragma unroll
        for (int pp = 0; pp < 4 / kParts; ++pp) tmem_ld32(tmem_row + kAccCol0 + as * kChunk + (h + kParts * pp) * 32, v[pp]);
        tmem_ld_wait();
        tc_fence_before_sync();
        __syncwarp();
        if (lane == 0) mbar_arrive_leader(&s.acc_empty[as]);     // scores are in registers: the stage is free
        if (threadIdx.x == 64 && cg < 8) DBGT(48 + cg)
#pragma unroll
        for (int pp = 0; pp < 4 / kParts; ++pp) {
          const int piece = c * (kChunk / 32) + h + kParts * pp;
#ifdef MAPL_DBG
          if (threadIdx.x == 64 && cg < 8 && pp == 1) DBGT(56 + cg)      // piece 0 of the chunk done
#endif
          const uint32_t h4 = sHn_u32 + piece * 128;      // explicit ld.shared: the carved pointers compile to generic loads
          float sc[32];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float4 hh;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(hh.x), "=f"(hh.y), "=f"(hh.z), "=f"(hh.w) : "r"(h4 + 16 * i));
            sc[4 * i + 0] = fmaf(__uint_as_float(v[pp][4 * i + 0]), nsc, hh.x);
            sc[4 * i + 1] = fmaf(__uint_as_float(v[pp][4 * i + 1]), nsc, hh.y);
            sc[4 * i + 2] = fmaf(__uint_as_float(v[pp][4 * i + 2]), nsc, hh.z);
            sc[4 * i + 3] = fmaf(__uint_as_float(v[pp][4 * i + 3]), nsc, hh.w);
          }
          // The min / compare instructions run on the half-rate ALU pipe, which bounds this loop at r = 64: three-input
          // minima, and the candidate mask from the sign bits of thr - sc (an FADD on the FMA pipe and one funnel
          // shift per codeword instead of FSETP + SEL + OR).
          float mn[4];
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            const float a = fminf(fminf(sc[8 * g], sc[8 * g + 1]), sc[8 * g + 2]);
            const float b = fminf(fminf(sc[8 * g + 3], sc[8 * g + 4]), sc[8 * g + 5]);
            mn[g] = fminf(fminf(a, b), fminf(sc[8 * g + 6], sc[8 * g + 7]));
          }
          const float m32 = fminf(fminf(mn[0], mn[1]), fminf(mn[2], mn[3]));
          best = fminf(best, m32);
          const float thr = best + margin;
          if (__any_sync(full, live && m32 <= thr)) {      // dead rows hold stale smem: never candidates
            // bit i of mask <=> sc[i] <= thr <=> sign(thr - sc[i]) clear (thr - sc == +0 when equal)
            uint32_t mk[4] = {0u, 0u, 0u, 0u};
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
              for (int i = 7; i >= 0; --i) mk[g] = __funnelshift_l(__float_as_uint(thr - sc[8 * g + i]), mk[g], 1);
            const uint32_t mask = ~(mk[0] | (mk[1] << 8) | (mk[2] << 16) | (mk[3] << 24));
            if (live && mask != 0) {
              if (cnt == kNE) {                 // list full: drop entries the tighter threshold excludes
                int j = 0;
                for (int e = 0; e < kNE; ++e) {
                  const float em = eM[e * kEpi];
                  if (em <= thr) { eM[j * kEpi] = em; eP[j * kEpi] = eP[e * kEpi]; eMask[j * kEpi] = eMask[e * kEpi]; ++j; }
                }
                cnt = j;
              }
              if (cnt == kNE) {
                // still full: the list keeps the kNE pieces with the lowest minima.  A piece left out matters only if
                // its minimum is within the FINAL threshold (checked after the scan; the threshold only tightens), so a
                // list that is full for a moment under the early, loose threshold no longer forces the exhaustive pass.
                int w = 0;
                float wm = eM[0];
                for (int e = 1; e < kNE; ++e) {
                  const float em = eM[e * kEpi];
                  if (em > wm) { wm = em; w = e; }
                }
                if (m32 < wm) {
                  dropped = fminf(dropped, wm);
                  eM[w * kEpi] = m32; eP[w * kEpi] = piece; eMask[w * kEpi] = mask;     // entries no longer ascend in k
                } else {
                  dropped = fminf(dropped, m32);
                }
              } else {
                eM[cnt * kEpi] = m32; eP[cnt * kEpi] = piece; eMask[cnt * kEpi] = mask; ++cnt;
              }
            }
          }
        }
      }
      xBest[mine] = best;
      epi_sync();
#pragma unroll
      for (int hh = 0; hh < kParts; ++hh) best = fminf(best, xBest[hh * 128 + row]);
      if (warp == 2 && l < 4) { DBG(5 + l * 4) }

      // ---- exact fp32 re-scoring of this thread's candidates: lowest score, lowest index on ties
      const float thr = best + margin;
      const bool overflow = live && dropped <= thr;     // pathological (e.g. many duplicate codewords): exhaustive below
      float bestx = FLT_MAX;
      int bestk = 0x7fffffff, e = 0, piece = 0;
      uint32_t mrem = 0;
      while (true) {
        while (mrem == 0 && e < cnt) {
          if (eM[e * kEpi] <= thr) { mrem = eMask[e * kEpi]; piece = eP[e * kEpi]; }
          ++e;
        }
        const bool have = mrem != 0 && !overflow;
        if (!__any_sync(full, have)) break;
        int k = 0;
        if (have) { k = piece * 32 + __ffs(mrem) - 1; mrem &= mrem - 1; }
        const float sx = exact_score(tmem_row, Cl + (long long)k * p.r, s.sHn[k], p.r);
        if (have && (sx < bestx || (sx == bestx && k < bestk))) { bestx = sx; bestk = k; }
      }
      if (__any_sync(full, overflow)) {         // exhaustive over the pieces this warp owns
        for (int pc = h; pc < p.K / 32; pc += kParts)
          for (int i = 0; i < 32; ++i) {
            const int k = pc * 32 + i;
            const float sx = exact_score(tmem_row, Cl + (long long)k * p.r, s.sHn[k], p.r);
            if (overflow && sx < bestx) { bestx = sx; bestk = k; }
          }
      }
      xScore[mine] = bestx; xK[mine] = bestk;
      epi_sync();
#pragma unroll
      for (int hh = 0; hh < kParts; ++hh) {
        const float ox = xScore[hh * 128 + row];
        const int ok = xK[hh * 128 + row];
        if (ox < bestx || (ox == bestx && ok < bestk)) { bestx = ox; bestk = ok; }
      }
      if (bestk == 0x7fffffff) bestk = 0;       // dead rows
#pragma unroll
      for (int ll = 0; ll < 8; ++ll) if (ll == l) code_l[ll] = bestk;
      if (warp == 2 && l < 4) { DBG(6 + l * 4) }
      if (live && h == 0) p.codes[m * p.L + l] = bestk;
      if (l + 1 < p.L) {
        rho_subtract(tmem_row, Cl + (long long)bestk * p.r, p.r, h, &n2, &amax);
        xN2[mine] = n2; xAmax[mine] = amax;
        epi_sync();
        n2 = 0.f; amax = 0.f;
#pragma unroll
        for (int hh = 0; hh < kParts; ++hh) { n2 += xN2[hh * 128 + row]; amax = fmaxf(amax, xAmax[hh * 128 + row]); }
        unscale = rho_to_operand(tmem_row, s.sRho, row, p.r, h, amax);
        fence_proxy_async_smem();
        tc_fence_before_sync();
        __syncwarp();
        if (lane == 0) mbar_arrive_leader(s.rho_ready);
      }
    }

    if (warp == 2) { DBG(2) }
    if (p.Zq != nullptr && live) {                          // zhat = sum_l C[l, code_l, :], rounded once
      for (int cc = h; cc < p.r / 8; cc += kParts) {
        float a[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int l = 0; l < 8; ++l) {
          if (l < p.L) {
            const float4* src = reinterpret_cast<const float4*>(p.C + ((long long)l * p.K + code_l[l]) * p.r + cc * 8);
            const float4 x = __ldg(src), y = __ldg(src + 1);
            a[0] += x.x; a[1] += x.y; a[2] += x.z; a[3] += x.w; a[4] += y.x; a[5] += y.y; a[6] += y.z; a[7] += y.w;
          }
        }
        *reinterpret_cast<uint4*>(p.Zq + m * p.r + cc * 8) =
            make_uint4(pack_bf16x2(a[0], a[1]), pack_bf16x2(a[2], a[3]), pack_bf16x2(a[4], a[5]), pack_bf16x2(a[6], a[7]));
      }
    }
  }
  tc_fence_before_sync();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc_pair<512>(tmem_base);
  }
}

}  // namespace
}  // namespace mapl
MAPL_DBG_READER(mapl_debug_read_rvq)
namespace mapl {

int tc_encode_rvq(const mapl_boundary_desc& d, const void* H, const float* codebooks, const TcPack& pk, void* Zq_out,
                  int32_t* codes_out, cudaStream_t st, const int32_t* tok, const float* Tc) {
  if (!tc_rvq_ok(d) || !pk.WBlo || !pk.Cb) return MAPL_ERR_UNSUPPORTED;
  RvqParams p;
  p.C = codebooks; p.hn = pk.hn; p.cmax = pk.cmax; p.cscale = pk.cscale; p.tok = tok; p.Tc = Tc;
  p.Zq = reinterpret_cast<__nv_bfloat16*>(Zq_out); p.codes = codes_out;
  p.N = d.n_tokens; p.d = d.d; p.r = d.r; p.L = d.rvq_levels; p.K = d.rvq_k;
  p.tile_m = tc_tile_m(d.n_tokens);
  p.stage1_bytes = kTileBytes + 2 * d.r * 64;
  p.stages1 = 2; p.ring_tiles = 2;
  const size_t avail = (size_t)227 * 1024 - 1024 - rvq_tail_bytes(p);
  if (avail < (size_t)2 * p.stage1_bytes || avail < (size_t)(d.r / 64 + 1) * kTileBytes) return MAPL_ERR_UNSUPPORTED;
  p.stages1 = (int)(avail / p.stage1_bytes);
  if (p.stages1 > 8) p.stages1 = 8;
  if (p.stages1 > d.d / 64) p.stages1 = d.d / 64;
  p.ring_tiles = (int)((avail - (size_t)(d.r / 64) * kTileBytes) / kHalfTileBytes);
  if (p.ring_tiles > 16) p.ring_tiles = 16;
  if (p.stages1 < 2 || p.ring_tiles < 2) return MAPL_ERR_UNSUPPORTED;
  const size_t smem = 1024 + rvq_regionR(p) + rvq_tail_bytes(p);
  CUtensorMap tmH, tmWhi, tmWlo, tmC;
  const uint64_t dd = (uint64_t)d.d, rr = (uint64_t)d.r;
  if (!make_tmap_bf16_2d(&tmH, H, (uint64_t)d.n_tokens, dd, dd, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmWhi, pk.WB, rr, dd, dd, 64, (uint32_t)d.r / 2)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmWlo, pk.WBlo, rr, dd, dd, 64, (uint32_t)d.r / 2)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmC, pk.Cb, (uint64_t)d.rvq_levels * d.rvq_k, rr, rr, 64, kChunk / 2)) return MAPL_ERR_CUDA;
  MAPL_SMEM_OPT_IN(k_tc_encode_rvq, 227 * 1024);
  const unsigned tiles = ((unsigned)((d.n_tokens + p.tile_m - 1) / p.tile_m) + 1u) & ~1u;   // whole CTA pairs
  KernelScope ks(KID_TC_ENCODE_RVQ, st);
  MAPL_CUDA_CHECK(launch_pdl_pair(k_tc_encode_rvq, dim3(tiles), dim3(kThreads), smem, st, tmH, tmWhi, tmWlo, tmC, p));
  return MAPL_OK;
}

}  // namespace mapl
