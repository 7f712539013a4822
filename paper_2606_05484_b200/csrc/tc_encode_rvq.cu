// tc_encode_rvq.cu -- mapl_encode with residual VQ on the tensor cores: projection and all RVQ
// levels in ONE kernel, z never leaves the chip (Eq. 1; Sec. 3.5;
// readings S3-S5, S18 of DESIGN.md).
//
// One CTA per token tile (<= 128 tokens; one TMEM lane = one token); CTAs work in pairs (cluster of 2,
// cta_group::2 MMAs of M = 256): each CTA loads half of every parameter / codebook tile.
//   phase 1   z = H (U_hi + U_lo [+ U_lo2])   H tiles by TMA (HBM, evict-first), the bf16 split terms of U^T from the
//             L2-resident pack; fp32 accumulator [128 x r] in TMEM columns [0,r).  bf16 H is exact; two terms carry 16
//             mantissa bits of U, three (L >= 3) all 24, so that the deep levels stay inside rule S5.
//   level l   rho (fp32) stays in TMEM columns [0,r); its fp16 rounding, scaled per token by a power of two inv, is the
//             resident A operand (the codebook copy is fp16 too, scaled per level by sc_l).  Codebook tiles
//             [128 codewords x 64] stream through a TMA ring; per 128-codeword chunk one accumulator stage
//                 T_k = rho_s . c_s,k  -  a' q_k        (2 stages, TMEM cols 256..511)
//             where the second term is ONE extra K = 16 MMA step: the A side holds a' = inv 2^g in all 16 columns, the
//             B side the three-term fp16 split of -q_k, q_k = 0.5 ||c_k||^2 sc_l 2^-g (SWIZZLE_32B tiles; a constant A
//             row makes the column order irrelevant).  T_k = inv sc_l (rho.c_k - 0.5||c_k||^2) up to the coarse error
//                 E = E_op + E_acc + E_hn   (fp16 operand rounding, tensor-core accumulation, the split of q)
//             so argmax_k T_k is the nearest codeword up to E.  Epilogue (2 threads per token, 64 scores per thread and
//             chunk): a max3 tree per 16-codeword group (0.5 instruction per score) and the running maximum; a group
//             whose maximum is within 2E of the running maximum is STASHED raw (four 16-byte stores) in a per-thread
//             list in shared memory.  After the scan the final threshold best - 2E prunes the list; the surviving
//             groups are re-read, their scores >= the threshold are the candidates (the true minimiser is always
//             among them); a token with a single candidate is done, the others are re-scored in exact fp32 in the
//             DIRECT form sum_j (rho_j - c_kj)^2 (rho from TMEM, the fp32 codeword from L2), lowest index winning
//             ties (S4).  Then rho -= C[l, k*], fused with the fp16 conversion for the next level (the scale comes
//             from the bound max|rho| + max|c|: fp16 precision does not depend on it).
//             A list holds kne groups in shared memory, written without branches as a FIFO (the threshold only rises,
//             so the oldest entry is the likeliest to be stale); a live entry that must make room moves to a global
//             overflow area, and only a maximum that finds no room there either and is within the FINAL threshold
//             sends the thread to the exhaustive fp32 pass over its codewords (duplicate-heavy codebooks).
// Roofline: tensor at config 3 (K r = 1M per level), HBM at config 2.
#include <float.h>

#include "profile.cuh"
#include "tc_codec.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

constexpr int kParts = 2;                // scan / re-score threads per token (warps per TMEM lane quarter)
constexpr int kEpi = 128 * kParts;       // epilogue threads
constexpr int kProducers = 3;            // TMA producer warps: warp 0 and the two warps after the epilogue warps.  A producer
                                         // thread pays ~560 cycles per loop iteration plus ~135 per 8 KB box whatever the ring depth
                                         // (measured: _work microbenchmark); the cost is per THREAD, so
                                         // several producer warps taking the items in turn multiply the issue rate
constexpr int kThreads = 64 + kEpi + 64; // warp 0 TMA, warp 1 MMA, kParts x 4 scan / re-score warps, 2 more TMA warps
constexpr int kChunk = 128;              // codewords per accumulator stage (UMMA N)
constexpr int kAccCol0 = 256;            // TMEM column of score stage 0
constexpr int kXStages = 8;              // ring of the norm tiles (one per chunk)
constexpr int kXBytes = 64 * 32;         // a CTA's half of a norm tile: 64 codewords x 16 fp16
constexpr int kAxBytes = 128 * 32;       // A side of the norm step: 128 tokens x 16 fp16

struct RvqParams {
  const float* C;        // [L,K,r] fp32 codebooks (exact re-scoring, residual update)
  const float* lvl;      // [8 x 8] per-level constants (tc_codec.cuh)
  const int32_t* tok; const float* Tc;   // optional sender-side centring (Eq. 1): z -= Tc[tok], Tc [V,r] fp32
  __nv_bfloat16* Zq;     // optional [N,r]
  int32_t* codes;        // [N,L]
  long long N;
  int d, r, L, K, tile_m;
  int stages1, stage1_bytes, ring_tiles, nsplit, kne, p1, p2;
  uint8_t* ovf; int kovf;   // global overflow entries per scan thread (tc_codec.cuh); kovf == 0: none
};

// smem carve-up (after 1024-byte alignment):
//   region R = max(phase-1 ring,  rho operand tiles | norm A tile | codebook ring | norm ring | stash)
//   eM [kne][kEpi] f32 | eId [kne][kEpi] i32 | exchange [6][kEpi] | xCand [kEpi][4] i32 | barriers | tmem slot
struct Smem {
  uint8_t* ring1; uint8_t* sRho; uint8_t* sAx; uint8_t* ringC; uint8_t* ringX; uint8_t* stash;
  float* eM; int* eId;
  float* xch;            // [6][kEpi]: best / dist / k / n2 / amax / count exchanged by the threads of a token
  int* xcand;            // [kEpi][4]: the first candidates of every thread, shared by the threads of a token
  uint64_t* s1_full; uint64_t* s1_empty; uint64_t* z_full;
  uint64_t* c_full; uint64_t* c_empty; uint64_t* x_full; uint64_t* x_empty;
  uint64_t* acc_full; uint64_t* acc_empty; uint64_t* rho_ready;
  uint32_t* tmem_slot;
};

__host__ __device__ inline size_t rvq_level_bytes(const RvqParams& p) {
  return (size_t)(p.r / 64) * kTileBytes + kAxBytes + (size_t)p.ring_tiles * kHalfTileBytes + (size_t)kXStages * kXBytes +
         (size_t)p.kne * 4 * kEpi * 16;
}
__host__ __device__ inline size_t rvq_regionR(const RvqParams& p) {
  const size_t ring1 = (size_t)p.stages1 * p.stage1_bytes, lvl = rvq_level_bytes(p);
  return ring1 > lvl ? ring1 : lvl;
}
__host__ __device__ inline size_t rvq_tail_bytes(int kne) {
  return (size_t)kne * kEpi * 8 + 6 * kEpi * 4 + kEpi * 4 * 4 + 1024;
}

__device__ __forceinline__ Smem carve_smem(uint8_t* base, const RvqParams& p) {
  Smem s;
  s.ring1 = base;
  s.sRho = base;
  s.sAx = s.sRho + (size_t)(p.r / 64) * kTileBytes;
  s.ringC = s.sAx + kAxBytes;
  s.ringX = s.ringC + (size_t)p.ring_tiles * kHalfTileBytes;
  s.stash = s.ringX + (size_t)kXStages * kXBytes;
  uint8_t* t = base + rvq_regionR(p);
  s.eM = reinterpret_cast<float*>(t); t += (size_t)p.kne * kEpi * 4;
  s.eId = reinterpret_cast<int*>(t); t += (size_t)p.kne * kEpi * 4;
  s.xch = reinterpret_cast<float*>(t); t += 6 * kEpi * 4;
  s.xcand = reinterpret_cast<int*>(t); t += kEpi * 4 * 4;
  uint64_t* b = reinterpret_cast<uint64_t*>(t);
  s.s1_full = b; b += p.stages1;
  s.s1_empty = b; b += p.stages1;
  s.z_full = b; b += 1;
  s.c_full = b; b += p.ring_tiles;
  s.c_empty = b; b += p.ring_tiles;
  s.x_full = b; b += kXStages;
  s.x_empty = b; b += kXStages;
  s.acc_full = b; b += 2;
  s.acc_empty = b; b += 2;
  s.rho_ready = b; b += 1;
  s.tmem_slot = reinterpret_cast<uint32_t*>(b);
  return s;
}

// exact fp32 squared distance of codeword row `crow` to this thread's residual (TMEM columns [0,r)), in the DIRECT
// form sum_j (rho_j - c_j)^2 the oracle uses (no cancellation when D << ||c||^2).  Warp-convergent (tcgen05.ld is
// .sync.aligned); lanes without work pass any valid row and ignore the result.
__device__ __forceinline__ float exact_dist(uint32_t tmem_row, const float* __restrict__ crow, int r) {
  // One 32-column piece of the row (8 float4, L2 latency) is in flight while the piece before it is consumed: the
  // pass costs one L2 round trip plus r / 32 short steps, where loading two pieces per round and then consuming them
  // cost r / 64 round trips (r is a multiple of 64: an even number of pieces).
  // Four accumulators (columns j = 0, 1, 2, 3 mod 4), summed as (a0 + a1) + (a2 + a3) at the end: one chain of r
  // dependent FMAs was ~1000 cycles of pure latency per candidate.  exhaustive_half sums in the same order.
  const float4* c4 = reinterpret_cast<const float4*>(crow);
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  float4 ca[8], cb[8];
  auto consume = [&](const float4 (&c)[8], int pc) {
    uint32_t v[32];
    tmem_ld32(tmem_row + pc * 32, v);
    tmem_ld_wait();
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float d0 = __uint_as_float(v[4 * i + 0]) - c[i].x, d1 = __uint_as_float(v[4 * i + 1]) - c[i].y;
      const float d2 = __uint_as_float(v[4 * i + 2]) - c[i].z, d3 = __uint_as_float(v[4 * i + 3]) - c[i].w;
      a0 = fmaf(d0, d0, a0); a1 = fmaf(d1, d1, a1); a2 = fmaf(d2, d2, a2); a3 = fmaf(d3, d3, a3);
    }
  };
#pragma unroll
  for (int i = 0; i < 8; ++i) ca[i] = __ldg(c4 + i);
  const int np = r / 32;
#pragma unroll 1
  for (int pc = 0; pc < np; pc += 2) {
#pragma unroll
    for (int i = 0; i < 8; ++i) cb[i] = __ldg(c4 + (pc + 1) * 8 + i);
    consume(ca, pc);
    if (pc + 2 < np) {
#pragma unroll
      for (int i = 0; i < 8; ++i) ca[i] = __ldg(c4 + (pc + 2) * 8 + i);
    }
    consume(cb, pc + 1);
  }
  return (a0 + a1) + (a2 + a3);
}

// The exhaustive pass for ONE token (the lane `owner` of this warp) over the codewords its thread owns: the 32-codeword
// pieces pc = h, h + kParts, ... of the level.  The owner's residual is handed to the warp piece by piece (shuffles) and
// lane j scores codeword j of every piece, four at a time, accumulating in exact_dist's order (so a distance has
// the same bits whichever path computed it: duplicate codewords tie exactly); the minimum (distance, then index) goes
// back to the owner.  ~40 us per token where the owner alone needed 2-4 ms (K / 2 serial passes with 31 lanes idle):
// the pass is rare (a token whose candidate lists ran out of room, once in ~3000 steps of the config 3 run) but it
// was visible as a 4 ms step.  Warp-convergent.
__device__ __forceinline__ void exhaustive_half(uint32_t tmem_row, const float* __restrict__ Cl, int r, int K, int h,
                                                int lane, int owner, float* bestx, int* bestk) {
  const unsigned full = 0xffffffffu;
  const int npieces = K / 32 / kParts;
  float bx = FLT_MAX;
  int bk = 0x7fffffff;
#pragma unroll 1
  for (int t0 = 0; t0 < npieces; t0 += 4) {
    float acc[4][4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { acc[u][0] = 0.f; acc[u][1] = 0.f; acc[u][2] = 0.f; acc[u][3] = 0.f; }
#pragma unroll 1
    for (int pc = 0; pc < r / 32; ++pc) {
      uint32_t v[32];
      tmem_ld32(tmem_row + pc * 32, v);
      tmem_ld_wait();
      float rb[32];
#pragma unroll
      for (int j = 0; j < 32; ++j) rb[j] = __shfl_sync(full, __uint_as_float(v[j]), owner);
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (t0 + u < npieces) {
          const int k = (h + kParts * (t0 + u)) * 32 + lane;
          const float4* c4 = reinterpret_cast<const float4*>(Cl + (long long)k * r + pc * 32);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float4 c = __ldg(c4 + i);
            const float d0 = rb[4 * i + 0] - c.x, d1 = rb[4 * i + 1] - c.y, d2 = rb[4 * i + 2] - c.z, d3 = rb[4 * i + 3] - c.w;
            acc[u][0] = fmaf(d0, d0, acc[u][0]); acc[u][1] = fmaf(d1, d1, acc[u][1]);
            acc[u][2] = fmaf(d2, d2, acc[u][2]); acc[u][3] = fmaf(d3, d3, acc[u][3]);
          }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int k = (h + kParts * (t0 + u)) * 32 + lane;
      const float dx = (acc[u][0] + acc[u][1]) + (acc[u][2] + acc[u][3]);
      if (t0 + u < npieces && (dx < bx || (dx == bx && k < bk))) { bx = dx; bk = k; }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ox = __shfl_xor_sync(full, bx, o);
    const int ok = __shfl_xor_sync(full, bk, o);
    if (ox < bx || (ox == bx && ok < bk)) { bx = ox; bk = ok; }
  }
  if (lane == owner && (bx < *bestx || (bx == *bestx && bk < *bestk))) { *bestx = bx; *bestk = bk; }
}

// power of two inv with A * inv in [0.5, 1) for the bound A >= max|rho_j| (A == 0 / denormal: inv = 1)
__device__ __forceinline__ float inv_scale_of(float A) {
  int eb = (int)((__float_as_uint(A) >> 23) & 0xffu);
  eb = eb < 2 ? 126 : (eb > 250 ? 250 : eb);
  return __uint_as_float((uint32_t)(253 - eb) << 23);
}

__device__ __forceinline__ void store_operand_piece(uint8_t* sRho, int row, int pc, const uint32_t (&v)[32], float inv) {
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

// The kParts threads of a token split the residual by 32-column pieces: part h owns the pieces pc with pc % kParts == h.
// Level 0: rho <- z (+ second accumulator: the two halves of the projection chain) (- sub: the centring row) on the own
// pieces; partial ||rho||^2 and max|rho_j| of those pieces.  Warp-convergent.
__device__ __forceinline__ void rho_first(uint32_t tmem_row, const float* __restrict__ sub, bool add_second, int r, int h,
                                          float* n2_out, float* amax_out) {
  float n2 = 0.f, amax = 0.f;
  for (int pc = h; pc < r / 32; pc += kParts) {
    uint32_t v[32];
    tmem_ld32(tmem_row + pc * 32, v);
    if (add_second) {
      uint32_t w[32];
      tmem_ld32(tmem_row + kAccCol0 + pc * 32, w);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) + __uint_as_float(w[i]));
    } else {
      tmem_ld_wait();
    }
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
    }
    if (sub != nullptr || add_second) tmem_st32(tmem_row + pc * 32, v);
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const float x = __uint_as_float(v[i]);
      n2 = fmaf(x, x, n2);
      amax = fmaxf(amax, fabsf(x));
    }
  }
  if (sub != nullptr || add_second) tmem_st_wait();
  *n2_out = n2; *amax_out = amax;
}

// Levels >= 1: rho <- rho - C[k*] on the own pieces (pc = h, h + kParts, ...) and, in the same pass, the fp16 rounding
// of rho * inv into the swizzled A-operand tiles.  The codeword segments are loaded CO-OPERATIVELY: eight lanes fetch the
// 128 bytes of one token's segment, so a load instruction touches 4 full lines; every lane fetching its own token's row
// touched 32 lines per instruction and the pass was bound by the L1 tag stage (4.6 us at config 3: ~3700 cycles for
// each round of 16 loads).  The segments go through a per-warp staging buffer (`stage`: 32 tokens x 144 bytes, the pad
// keeps the 16-byte accesses conflict-free) to the lane that owns the token.  k is the lane's chosen codeword (any valid
// index on dead rows).  Warp-convergent.
constexpr int kStagePitch = 144;
__device__ __forceinline__ void rho_update(uint32_t tmem_row, const float* __restrict__ Cl, int k, uint8_t* sRho, uint8_t* stage,
                                           int row, int r, int h, int lane, float inv, float* n2_out, float* amax_out) {
  const unsigned full = 0xffffffffu;
  float n2 = 0.f, amax = 0.f;
  const int npc = r / 32 / kParts;
  const float* rowp[8];                                  // this lane's share of the fetches: token 4 j + lane / 8, chunk lane % 8
#pragma unroll
  for (int j = 0; j < 8; ++j) rowp[j] = Cl + (long long)__shfl_sync(full, k, 4 * j + lane / 8) * r + (lane % 8) * 4;
#pragma unroll 1
  for (int i = 0; i < npc; ++i) {
    const int pc = h + i * kParts;
    float4 x[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = __ldg(reinterpret_cast<const float4*>(rowp[j] + pc * 32));
#pragma unroll
    for (int j = 0; j < 8; ++j)
      *reinterpret_cast<float4*>(stage + (4 * j + lane / 8) * kStagePitch + (lane % 8) * 16) = x[j];
    __syncwarp();
    float4 c[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) c[j] = *reinterpret_cast<const float4*>(stage + lane * kStagePitch + j * 16);
    __syncwarp();
    uint32_t v[32];
    tmem_ld32(tmem_row + pc * 32, v);
    tmem_ld_wait();
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      v[4 * j + 0] = __float_as_uint(__uint_as_float(v[4 * j + 0]) - c[j].x);
      v[4 * j + 1] = __float_as_uint(__uint_as_float(v[4 * j + 1]) - c[j].y);
      v[4 * j + 2] = __float_as_uint(__uint_as_float(v[4 * j + 2]) - c[j].z);
      v[4 * j + 3] = __float_as_uint(__uint_as_float(v[4 * j + 3]) - c[j].w);
    }
    tmem_st32(tmem_row + pc * 32, v);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const float xv = __uint_as_float(v[j]);
      n2 = fmaf(xv, xv, n2);
      amax = fmaxf(amax, fabsf(xv));
    }
    store_operand_piece(sRho, row, pc, v, inv);
  }
  tmem_st_wait();
  *n2_out = n2; *amax_out = amax;
}

// fp16 conversion alone (level 0, once the exact max|z_j| of the token is known)
__device__ __forceinline__ void rho_to_operand(uint32_t tmem_row, uint8_t* sRho, int row, int r, int h, float inv) {
  for (int pc = h; pc < r / 32; pc += kParts) {
    uint32_t v[32];
    tmem_ld32(tmem_row + pc * 32, v);
    tmem_ld_wait();
    store_operand_piece(sRho, row, pc, v, inv);
  }
}

// named barrier 1 over the epilogue warps
__device__ __forceinline__ void epi_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kEpi) : "memory"); }

// maximum of 16 scores: 8 three-input maxima
__device__ __forceinline__ float max16(const uint32_t* v) {
#define MAPL_F(i) __uint_as_float(v[i])
  const float a = fmaxf(fmaxf(MAPL_F(0), MAPL_F(1)), MAPL_F(2)), b = fmaxf(fmaxf(MAPL_F(3), MAPL_F(4)), MAPL_F(5));
  const float c = fmaxf(fmaxf(MAPL_F(6), MAPL_F(7)), MAPL_F(8)), d = fmaxf(fmaxf(MAPL_F(9), MAPL_F(10)), MAPL_F(11));
  const float e = fmaxf(fmaxf(MAPL_F(12), MAPL_F(13)), MAPL_F(14));
  const float f = MAPL_F(15);
#undef MAPL_F
  return fmaxf(fmaxf(fmaxf(a, b), c), fmaxf(fmaxf(d, e), f));
}

// explicit shared-space accesses (pointers carved from the dynamic buffer compile to generic LD / ST otherwise)
__device__ __forceinline__ float lds_f32(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ int lds_s32(uint32_t a) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint4 lds_v4(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_s32(uint32_t a, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_v4(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

// per-thread candidate list.  Entries [0, kne) live in shared memory: entry e of thread t has its maximum at
// eM[e * kEpi + t], its group id (codeword index / 16) at eId[...], its 16 raw scores as four 16-byte units at
// stash[((e * 4 + i) * kEpi + t) * 16] (consecutive lanes -> consecutive 16-byte units: conflict-free).  Entries
// [kne, kne + kovf) live in the thread's slice of a global overflow area (80 bytes each: m, id, pad, pad, 16 scores),
// written only by the rare token with more than kne groups within its margin (measured at config 3: at most 7
// candidates per token, i.e. a handful of tokens per launch -- which cost 4 ms each when the list simply overflowed
// into the exhaustive pass).
struct CandList {
  uint32_t eM, eId, stash;   // shared-space byte addresses, already offset by the thread index
  uint8_t* ovf;              // this thread's global overflow entries (nullptr: none)
  int kne, kovf;
  int cnt;             // shared-memory entries in use (high-water mark)
  int slot;            // next slot of the FIFO
  int novf;            // overflow entries in use
  float dropped;       // highest maximum that found no room anywhere (-FLT_MAX: none)
};

__device__ __forceinline__ void ovf_put(CandList& cl, float m, int gid, const uint4 (&q)[4]) {
  if (cl.novf < cl.kovf) {
    uint4* e = reinterpret_cast<uint4*>(cl.ovf + (size_t)cl.novf * kRvqOverflowBytes);
    e[0] = make_uint4(__float_as_uint(m), (uint32_t)gid, 0u, 0u);
#pragma unroll
    for (int i = 0; i < 4; ++i) e[1 + i] = q[i];
    ++cl.novf;
  } else {
    cl.dropped = fmaxf(cl.dropped, m);
  }
}

// predicated shared-memory accesses: the scan appends to its list WITHOUT branches.  With one token per lane nearly
// every chunk has some lane whose group is within the margin (a running maximum is beaten ~ln(groups) times per level,
// times 32 lanes), so a branchy append ran its whole body for every group of every chunk: 130 of the loop's 162
// warp-instructions, each paying its full latency with two warps per scheduler (ncu source page, config 2: 12 % of
// the loop's samples issue, the rest are `wait` / `branch_resolving`) -- the scan was bound by this code, not by the
// TMEM read-out (the earlier 57 B/cycle read-out figure was an artefact of a microbenchmark that spilled to local memory).
__device__ __forceinline__ float lds_f32_if(bool pr, uint32_t a, float other) {
  float v;
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\nmov.f32 %0, %3;\n@q ld.shared.f32 %0, [%1];\n}"
               : "=f"(v) : "r"(a), "r"((int)pr), "f"(other));
  return v;
}
// entry `slot` := (m, gid, 16 raw scores v[0..16)) if pr
__device__ __forceinline__ void sts_entry_if(bool pr, const CandList& cl, int slot, float m, int gid, const uint32_t* v) {
  const uint32_t aM = cl.eM + (uint32_t)slot * kEpi * 4, aId = cl.eId + (uint32_t)slot * kEpi * 4;
  const uint32_t aS = cl.stash + (uint32_t)slot * 4 * kEpi * 16;
  asm volatile(
      "{\n.reg .pred q;\nsetp.ne.b32 q, %0, 0;\n"
      "@q st.shared.f32 [%1], %2;\n"
      "@q st.shared.s32 [%3], %4;\n"
      "@q st.shared.v4.u32 [%5], {%6, %7, %8, %9};\n"
      "@q st.shared.v4.u32 [%5 + 4096], {%10, %11, %12, %13};\n"
      "@q st.shared.v4.u32 [%5 + 8192], {%14, %15, %16, %17};\n"
      "@q st.shared.v4.u32 [%5 + 12288], {%18, %19, %20, %21};\n}"
      ::"r"((int)pr), "r"(aM), "f"(m), "r"(aId), "r"(gid), "r"(aS),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
        "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
      : "memory");
}
static_assert(kEpi * 16 == 4096, "sts_entry_if hard-codes the stride between the 16-byte units of an entry");

// The four 16-codeword groups of one chunk (maxima g[], ids gid[], raw scores v[i]) join the list where they are within
// the current threshold.  The shared-memory entries are a FIFO over kne >= 4 slots: the threshold only rises during a
// scan, so the oldest entry is the likeliest to be stale (below the threshold: droppable); if it is not, it moves to the
// global overflow entries first -- the one rare, divergent path, entered on a warp vote.  What finds no room there
// either is remembered in `dropped`, and only if that value is within the FINAL threshold does the thread need the
// exhaustive pass.
__device__ __forceinline__ void stash_chunk(CandList& cl, const float (&g)[4], const int (&gid)[4],
                                            const uint32_t* const (&v)[4], float thr, bool live) {
  bool pr[4], spill[4];
  int sl[4];
  bool any_spill = false;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    pr[i] = live && g[i] >= thr;
    sl[i] = cl.slot;
    const bool full = pr[i] && cl.cnt >= cl.kne;          // the slot holds an older entry
    const float m_old = lds_f32_if(full, cl.eM + (uint32_t)cl.slot * kEpi * 4, -FLT_MAX);
    spill[i] = full && m_old >= thr;
    any_spill |= spill[i];
    if (pr[i]) {
      cl.slot = cl.slot + 1 == cl.kne ? 0 : cl.slot + 1;
      cl.cnt = min(cl.cnt + 1, cl.kne);
    }
  }
  if (__any_sync(0xffffffffu, any_spill)) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
      if (spill[i]) {
        uint4 q[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) q[u] = lds_v4(cl.stash + (uint32_t)(sl[i] * 4 + u) * kEpi * 16);
        ovf_put(cl, lds_f32(cl.eM + (uint32_t)sl[i] * kEpi * 4), lds_s32(cl.eId + (uint32_t)sl[i] * kEpi * 4), q);
      }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) sts_entry_if(pr[i], cl, sl[i], g[i], gid[i], v[i]);
}

// entry e of the whole list (shared memory first, then the overflow entries): its maximum, group id, and the 16-bit
// mask of its scores >= thr
__device__ __forceinline__ float entry_max(const CandList& cl, int e) {
  if (e < cl.kne) return lds_f32(cl.eM + e * kEpi * 4);
  return __uint_as_float(reinterpret_cast<const uint4*>(cl.ovf + (size_t)(e - cl.kne) * kRvqOverflowBytes)[0].x);
}
__device__ __forceinline__ int entry_gid(const CandList& cl, int e) {
  if (e < cl.kne) return lds_s32(cl.eId + e * kEpi * 4);
  return (int)reinterpret_cast<const uint4*>(cl.ovf + (size_t)(e - cl.kne) * kRvqOverflowBytes)[0].y;
}
__device__ __forceinline__ uint32_t entry_mask(const CandList& cl, int e, float thr) {
  uint32_t mk = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint4 q = e < cl.kne ? lds_v4(cl.stash + (uint32_t)(e * 4 + i) * kEpi * 16)
                               : reinterpret_cast<const uint4*>(cl.ovf + (size_t)(e - cl.kne) * kRvqOverflowBytes)[1 + i];
    mk |= (__uint_as_float(q.x) >= thr ? 1u : 0u) << (4 * i);
    mk |= (__uint_as_float(q.y) >= thr ? 1u : 0u) << (4 * i + 1);
    mk |= (__uint_as_float(q.z) >= thr ? 1u : 0u) << (4 * i + 2);
    mk |= (__uint_as_float(q.w) >= thr ? 1u : 0u) << (4 * i + 3);
  }
  return mk;
}
// number of list positions to visit: all kne shared-memory positions once the overflow entries are in use
__device__ __forceinline__ int entry_count(const CandList& cl) { return cl.novf > 0 ? cl.kne + cl.novf : cl.cnt; }

__global__ void __launch_bounds__(kThreads, 1)
k_tc_encode_rvq(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmWhi,
                const __grid_constant__ CUtensorMap tmWlo, const __grid_constant__ CUtensorMap tmWlo2,
                const __grid_constant__ CUtensorMap tmC, const __grid_constant__ CUtensorMap tmX, const RvqParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const Smem s = carve_smem(smem, p);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t rank = cluster_ctarank();
  const long long m0 = (long long)blockIdx.x * p.tile_m;
  const int nkb1 = p.d / 64, nkb = p.r / 64, nchunks = p.K / kChunk;
  // Every CTA pair walks the codebook chunks (and the k-blocks of the projection) in its own rotation.  With one common
  // order all 74 pairs request the SAME L2 lines at the same moment and the requests serialise in the L2 slices that
  // hold them (measured at config 2: 2 us from TMA issue to arrival for an 8 KB L2-resident tile).  The arg-min does not
  // depend on the scan order (ties are decided on the codeword index in the exact pass).
  const int pair = blockIdx.x >> 1;
  const int rot_c = (int)(((unsigned)pair * 5u) % (unsigned)nchunks), rot_k = (int)(((unsigned)pair * 7u) % (unsigned)nkb1);

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmH); tma_prefetch_desc(&tmWhi); tma_prefetch_desc(&tmWlo); tma_prefetch_desc(&tmWlo2);
    tma_prefetch_desc(&tmC); tma_prefetch_desc(&tmX);
    for (int i = 0; i < p.stages1; ++i) { mbar_init(&s.s1_full[i], 1); mbar_init(&s.s1_empty[i], 1); }
    mbar_init(s.z_full, 1);
    for (int i = 0; i < p.ring_tiles; ++i) { mbar_init(&s.c_full[i], 1); mbar_init(&s.c_empty[i], 1); }
    for (int i = 0; i < kXStages; ++i) { mbar_init(&s.x_full[i], 1); mbar_init(&s.x_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s.acc_full[i], 1); mbar_init(&s.acc_empty[i], 8 * kParts); }
    mbar_init(s.rho_ready, 8 * kParts);               // leader's barriers collect the epilogue warps of both CTAs
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc_pair<512>(s.tmem_slot);
  // Rows tile_m .. 127 of the H tiles are never written by TMA (its box has tile_m rows) and are multiplied all the
  // same: zero them once, and give the dead rows a zero fp16 operand in the scans too (inv = 0 below).  The chip is
  // power-limited under tensor load and zero operands are cheap: c3 194.0 -> 192.5 us; it also
  // keeps whatever the previous kernel left in shared memory (NaN patterns included) out of the tensor pipe.
  if (p.tile_m < 128) {
    const int per_stage = (128 - p.tile_m) * 8;                       // 16-byte units of the dead rows of one H tile
    for (int i = threadIdx.x; i < p.stages1 * per_stage; i += kThreads) {
      const int st = i / per_stage, u = i - st * per_stage;
      *reinterpret_cast<uint4*>(s.ring1 + (size_t)st * p.stage1_bytes + (size_t)p.tile_m * 128 + (size_t)u * 16) = make_uint4(0u, 0u, 0u, 0u);
    }
    fence_proxy_async_smem();
  }
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem_base = *s.tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");       // everything below touches global memory
  if (warp == 0) { DBG(0) }

  if (warp == 0 || warp >= 2 + 4 * kParts) {
    // ------------------------------------------------------------ TMA producers: items (stages) in turn
    const int pi = warp == 0 ? 0 : warp - (1 + 4 * kParts);
    if (elect_one()) {
      const uint32_t w_tile = (uint32_t)p.r * 64;          // this CTA's half (r/2 rows) of a U^T tile
      const uint32_t tx1 = 2u * ((uint32_t)(p.tile_m * 128) + (uint32_t)p.nsplit * w_tile);
      const int wrow = (int)rank * (p.r / 2);
      // producers in use per phase: a producer may run at most ONE use of a ring slot ahead of the consumer (the
      // barriers carry one phase bit), which holds when the producers' items together fit the ring
      const int kP1 = p.p1, kP2 = p.p2;
      RingPos r1;
      r1.advance(pi, p.stages1);
      int kr = pi + rot_k;
      if (kr >= nkb1) kr -= nkb1;
#ifdef MAPL_DBG
      long long w_empty1 = 0;
#endif
      for (int kb = pi < kP1 ? pi : nkb1; kb < nkb1; kb += kP1) {
#ifdef MAPL_DBG
        const long long t_w = clock64();
#endif
        mbar_wait(&s.s1_empty[r1.st], r1.ph ^ 1u);
#ifdef MAPL_DBG
        w_empty1 += clock64() - t_w;
#endif
        if (rank == 0) mbar_arrive_expect_tx(&s.s1_full[r1.st], tx1);
        uint8_t* a = s.ring1 + (size_t)r1.st * p.stage1_bytes;
        tma_load_2d_pair(a, &tmH, &s.s1_full[r1.st], kr * 64, (int)m0, kEvictFirst);
        tma_load_2d_pair(a + kTileBytes, &tmWhi, &s.s1_full[r1.st], kr * 64, wrow, kEvictLast);
        tma_load_2d_pair(a + kTileBytes + w_tile, &tmWlo, &s.s1_full[r1.st], kr * 64, wrow, kEvictLast);
        if (p.nsplit == 3) tma_load_2d_pair(a + kTileBytes + 2 * w_tile, &tmWlo2, &s.s1_full[r1.st], kr * 64, wrow, kEvictLast);
        r1.advance(kP1, p.stages1);
        kr += kP1;
        if (kr >= nkb1) kr -= nkb1;
      }
#ifdef MAPL_DBG
      if (pi == 0) g_dbg[blockIdx.x * 64 + 23] = (unsigned long long)w_empty1;   // producer 0: cycles waiting for free stages
#endif
      mbar_wait(s.z_full, 0);             // phase-1 MMAs have consumed region R: it may be reused
      // level phase: producer pi takes the chunks pi, pi + kProducers, ... (counted over all levels): the chunk's nkb
      // codebook tiles and its norm tile
      RingPos rc, rx;
      rc.advance(pi * nkb, p.ring_tiles);
      rx.advance(pi, kXStages);
      int c = pi, l = pi < kP2 ? 0 : p.L;
      while (c >= nchunks) { c -= nchunks; ++l; }
      while (l < p.L) {
        int cr = c + rot_c;
        if (cr >= nchunks) cr -= nchunks;
        const int row0 = l * p.K + cr * kChunk + (int)rank * (kChunk / 2);
        RingPos t = rc;
        for (int j = 0; j < nkb; ++j) {
          mbar_wait(&s.c_empty[t.st], t.ph ^ 1u);
          if (rank == 0) mbar_arrive_expect_tx(&s.c_full[t.st], 2 * kHalfTileBytes);
          tma_load_2d_pair(s.ringC + (size_t)t.st * kHalfTileBytes, &tmC, &s.c_full[t.st], j * 64, row0, kEvictLast);
          t.next(p.ring_tiles);
        }
        mbar_wait(&s.x_empty[rx.st], rx.ph ^ 1u);
        if (rank == 0) mbar_arrive_expect_tx(&s.x_full[rx.st], 2 * kXBytes);
        tma_load_2d_pair(s.ringX + (size_t)rx.st * kXBytes, &tmX, &s.x_full[rx.st], 0, row0, kEvictLast);
        rc.advance(kP2 * nkb, p.ring_tiles);
        rx.advance(kP2, kXStages);
        c += kP2;
        while (c >= nchunks) { c -= nchunks; ++l; }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer
    if (rank == 0 && elect_one()) {
      const uint32_t idesc1 = make_idesc_bf16(256, (uint32_t)p.r, false, false);
      RingPos r1;
#ifdef MAPL_DBG
      long long w_full1 = 0;
#endif
      for (int kb = 0; kb < nkb1; ++kb) {
#ifdef MAPL_DBG
        const long long t_w = clock64();
#endif
        mbar_wait(&s.s1_full[r1.st], r1.ph);
#ifdef MAPL_DBG
        w_full1 += clock64() - t_w;
#endif
        tc_fence_after_sync();
        const uint32_t a = smem_u32(s.ring1 + (size_t)r1.st * p.stage1_bytes);
        const uint32_t bh = a + kTileBytes, bl = bh + p.r * 64, bl2 = bl + p.r * 64;
        // even / odd k-blocks accumulate into two TMEM regions ([0,r) and the still unused score stages at
        // [256,256+r)): the tensor core truncates when it adds into its accumulator, and halving the chain of
        // MMAs halves that one-sided error of z (tc_stiefel.cu measures it); the epilogue adds the two halves
        const uint32_t acc = tmem_base + (uint32_t)(kb & 1) * kAccCol0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint64_t da = desc_kmajor_sw128(a + k * 32);
          umma_bf16_pair(acc, da, desc_kmajor_sw128(bh + k * 32), idesc1, (kb >= 2) || k != 0);
          umma_bf16_pair(acc, da, desc_kmajor_sw128(bl + k * 32), idesc1, 1);
          if (p.nsplit == 3) umma_bf16_pair(acc, da, desc_kmajor_sw128(bl2 + k * 32), idesc1, 1);
        }
        umma_commit_pair(&s.s1_empty[r1.st]);
        r1.next(p.stages1);
      }
      umma_commit_pair(s.z_full);
#ifdef MAPL_DBG
      g_dbg[blockIdx.x * 64 + 22] = (unsigned long long)w_full1;      // cycles the projection MMAs waited for their stages
#endif
      const uint32_t idesc2 = make_idesc_f16(256, kChunk);
      const uint64_t dax = desc_kmajor_sw32_k16(smem_u32(s.sAx));
      const uint32_t ringX0 = smem_u32(s.ringX);
      const uint32_t la0 = desc_lo_kmajor_sw128(smem_u32(s.sRho)), lb0 = desc_lo_kmajor_sw128(smem_u32(s.ringC));
      RingPos rc, rx;
      uint32_t as = 0, aph = 0;            // accumulator stage and its use parity
      int cg = 0;
      for (int l = 0; l < p.L; ++l) {
        mbar_wait_cluster(s.rho_ready, l & 1);    // fp16 residuals of level l are in sRho / sAx of both CTAs
        tc_fence_after_sync();
        for (int c = 0; c < nchunks; ++c, ++cg) {
          mbar_wait_cluster(&s.acc_empty[as], aph ^ 1u);
          if (cg < 8) DBGT(24 + cg)
          tc_fence_after_sync();
          const uint32_t tmem_d = tmem_base + kAccCol0 + as * kChunk;
          for (int kb = 0; kb < nkb; ++kb) {
            mbar_wait(&s.c_full[rc.st], rc.ph);
            tc_fence_after_sync();
            const uint32_t a = la0 + (uint32_t)kb * (kTileBytes >> 4), b = lb0 + (uint32_t)rc.st * (kHalfTileBytes >> 4);
#pragma unroll
            for (int k = 0; k < 4; ++k) umma_bf16_pair_lo(tmem_d, a + 2 * k, b + 2 * k, idesc2, (kb | k) != 0);
            umma_commit_pair(&s.c_empty[rc.st]);
            rc.next(p.ring_tiles);
          }
          mbar_wait(&s.x_full[rx.st], rx.ph);       // + a' * (-q_k): the half norms, one K = 16 step
          tc_fence_after_sync();
          umma_bf16_pair(tmem_d, dax, desc_kmajor_sw32_k16(ringX0 + (uint32_t)rx.st * kXBytes), idesc2, 1);
          umma_commit_pair(&s.x_empty[rx.st]);
          umma_commit_pair(&s.acc_full[as]);
          rx.next(kXStages);
          if (cg < 8) DBGT(32 + cg)
          as ^= 1u;
          if (as == 0) aph ^= 1u;
        }
      }
    }
  } else {
    // ------------------------------------------------------------ epilogue: 4 kParts warps, kParts threads per token
    // q = TMEM lane quarter, h = which part of the 32-codeword pieces / 32-column pieces this warp owns
    const int q = warp & 3, h = (warp - 2) >> 2, row = q * 32 + lane;
    const long long m = m0 + row;
    const bool live = row < p.tile_m && m < p.N;
    const uint32_t tmem_row = tmem_base + ((uint32_t)(q * 32) << 16);
    const unsigned full = 0xffffffffu;
    float* xBest = s.xch; float* xDist = s.xch + kEpi; int* xK = reinterpret_cast<int*>(s.xch + 2 * kEpi);
    float* xN2 = s.xch + 3 * kEpi; float* xAmax = s.xch + 4 * kEpi; int* xCnt = reinterpret_cast<int*>(s.xch + 5 * kEpi);
    const int mine = h * 128 + row;
    CandList cl;
    cl.eM = smem_u32(s.eM + mine); cl.eId = smem_u32(s.eId + mine); cl.stash = smem_u32(s.stash) + (uint32_t)mine * 16;
    cl.kne = p.kne; cl.kovf = p.ovf != nullptr ? p.kovf : 0;
    cl.ovf = p.ovf != nullptr ? p.ovf + ((size_t)blockIdx.x * kEpi + mine) * (size_t)p.kovf * kRvqOverflowBytes : nullptr;
    int code_l[8];
#pragma unroll
    for (int l = 0; l < 8; ++l) code_l[l] = 0;
    const float sqrt_r = sqrtf((float)p.r), n_steps = (float)(p.r / 16 + 1);

    // the norm step's A row of this token: a' in all 16 columns (0 when a' is not an fp16 power of two: `hard` token)
    auto write_ax = [&](float ax, bool& hard) {
      hard = !(ax >= 5.9604645e-8f && ax <= 32768.f);
      if (h == 0) {
        const uint32_t w = pack_f16x2(hard ? 0.f : ax, hard ? 0.f : ax);
        uint4* dst = reinterpret_cast<uint4*>(s.sAx + (size_t)row * 32);
        dst[0] = make_uint4(w, w, w, w);
        dst[1] = make_uint4(w, w, w, w);
      }
    };
    auto publish_operand = [&]() {     // sRho / sAx rows of this warp are written: hand them to the MMA issuer
      fence_proxy_async_smem();
      tc_fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive_leader(s.rho_ready);
    };

    mbar_wait(s.z_full, 0);
    if (warp == 2) { DBG(1) }
    tc_fence_after_sync();
    float n2, amax, inv;
    bool hard;
    {
      // z = even-k-block half + odd-k-block half (see the MMA issuer), minus the centring row: the first residual is
      // z - Tc[tok] (dead rows subtract row 0: any valid row keeps the warp convergent)
      const float* csub = p.Tc != nullptr ? p.Tc + (live ? (long long)__ldg(p.tok + m) * p.r : 0) : nullptr;
      float n2p, amaxp;
      rho_first(tmem_row, csub, nkb1 >= 2, p.r, h, &n2p, &amaxp);
      xN2[mine] = n2p; xAmax[mine] = amaxp;
      epi_sync();
      n2 = 0.f; amax = 0.f;
#pragma unroll
      for (int hh = 0; hh < kParts; ++hh) { n2 += xN2[hh * 128 + row]; amax = fmaxf(amax, xAmax[hh * 128 + row]); }
      inv = inv_scale_of(amax);
      rho_to_operand(tmem_row, s.sRho, row, p.r, h, live ? inv : 0.f);
      write_ax(inv * __ldg(p.lvl + 2), hard);
      publish_operand();
    }

    int cg = 0;
#pragma unroll 1
    for (int l = 0; l < p.L; ++l) {
      const float* Cl = p.C + (long long)l * p.K * p.r;
      const float* lv = p.lvl + 8 * l;
      if (warp == 2 && l < 4) { DBG(4 + l * 4) }
      // 2E in the scaled units of T (file header): operand rounding, accumulation, the split of q
      float margin;
      {
        const float cmax_s = __ldg(lv), qmax = __ldg(lv + 1), ax = inv * __ldg(lv + 2);
        const float rs = sqrtf(n2) * inv;
        const float smax = rs * cmax_s + ax * qmax;
        const float e_op = 9.765625e-4f * 1.002f * rs * cmax_s + 2.9802322e-8f * sqrt_r * (cmax_s + rs);
        const float e_acc = n_steps * 1.9073486e-6f * (smax + 1.f);
        const float e_hn = ax * (1.1641532e-10f * qmax + 2.9802322e-8f);
        margin = 2.02f * (e_op + e_acc + e_hn);
      }

      float best = -FLT_MAX;
      cl.cnt = 0; cl.slot = 0; cl.novf = 0; cl.dropped = -FLT_MAX;
      int cr = rot_c;
      for (int c = 0; c < nchunks; ++c, ++cg) {
        const int as = cg & 1;
        mbar_wait(&s.acc_full[as], (cg >> 1) & 1);
        if (threadIdx.x == 64 && cg < 8) DBGT(40 + cg)
        tc_fence_after_sync();
        uint32_t v[2][32];            // this warp's pieces of the chunk: h and h + kParts
        tmem_ld32(tmem_row + kAccCol0 + as * kChunk + h * 32, v[0]);
        tmem_ld32(tmem_row + kAccCol0 + as * kChunk + (h + kParts) * 32, v[1]);
        tmem_ld_wait();
        tc_fence_before_sync();
        __syncwarp();
        if (lane == 0) mbar_arrive_leader(&s.acc_empty[as]);     // scores are in registers: the stage is free
        if (threadIdx.x == 64 && cg < 8) DBGT(48 + cg)
        const float g0 = max16(&v[0][0]), g1 = max16(&v[0][16]), g2 = max16(&v[1][0]), g3 = max16(&v[1][16]);
        const float m64 = fmaxf(fmaxf(g0, g1), fmaxf(g2, g3));
        best = fmaxf(best, m64);
        const float thr = best - margin;
        // dead rows hold stale data: never candidates
        {
          const int gid0 = (cr * 4 + h) * 2;               // 16-codeword group of v[0][0]; v[1] is kParts pieces further
          const float g[4] = {g0, g1, g2, g3};
          const int gid[4] = {gid0, gid0 + 1, gid0 + 2 * kParts, gid0 + 2 * kParts + 1};
          const uint32_t* const vv[4] = {&v[0][0], &v[0][16], &v[1][0], &v[1][16]};
          stash_chunk(cl, g, gid, vv, thr, live);
        }
        if (++cr == nchunks) cr = 0;
#ifndef MAPL_DBG2
        if (threadIdx.x == 64 && cg < 8) DBGT(56 + cg)
#endif
      }
      xBest[mine] = best;
      epi_sync();
#pragma unroll
      for (int hh = 0; hh < kParts; ++hh) best = fmaxf(best, xBest[hh * 128 + row]);
      if (warp == 2 && l < 4) { DBG(5 + l * 4) }

      // ---- candidates: every stashed score within the final threshold
      const float thr = best - margin;
      const bool overflow = live && (hard || cl.dropped >= thr);     // pathological (e.g. many duplicate codewords)
      int ncand = 0, firstk = 0;
      const int n_ent = entry_count(cl);
      for (int e = 0; e < n_ent; ++e) {
        if (entry_max(cl, e) >= thr) {
          const int k0 = entry_gid(cl, e) * 16;
          for (uint32_t mk = entry_mask(cl, e, thr); mk != 0; mk &= mk - 1) {
            const int k = k0 + __ffs(mk) - 1;
            if (ncand == 0) firstk = k;
            if (ncand < 4) s.xcand[mine * 4 + ncand] = k;     // the partner thread may take some of them (below)
            ++ncand;
          }
        }
      }
      if (!live) ncand = 0;
      xCnt[mine] = overflow ? 1000 : ncand;
#ifdef MAPL_DBG2
      atomicAdd(&g_dbg[blockIdx.x * 64 + 61], (unsigned long long)ncand);
      atomicAdd(&g_dbg[blockIdx.x * 64 + 60], (unsigned long long)n_ent);
      if (cl.novf) atomicAdd(&g_dbg[blockIdx.x * 64 + 59], (unsigned long long)cl.novf);
#endif
      epi_sync();
      if (warp == 2 && l < 4) { DBG(7 + l * 4) }
      static_assert(kParts == 2, "the balanced exact pass below is written for two threads per token");
      const int n0 = xCnt[row], n1 = xCnt[128 + row];
      const int tot = n0 + n1;
      // a single candidate is the minimiser (it is always among the candidates); else exact fp32 re-scoring,
      // lowest distance, lowest index on ties
      const bool rescore = tot >= 2;
      float bestx = FLT_MAX;
      int bestk = 0x7fffffff;
      if (!rescore && ncand == 1) { bestx = -1.f; bestk = firstk; }
      // The exact pass costs a warp as many serial passes as its busiest lane has candidates, so the two threads of a
      // token share the token's candidates: thread h takes numbers h, h + 2, ... of the joint list (the first four of
      // each thread are in shared memory).  A token with more than four in one thread keeps the per-thread pass.
      const bool balanced = rescore && tot < 1000 && n0 <= 4 && n1 <= 4;
      for (int i = h;; i += kParts) {
        const bool have = balanced && live && i < tot;
        if (!__any_sync(full, have)) break;
        const int k = have ? (i < n0 ? s.xcand[row * 4 + i] : s.xcand[(128 + row) * 4 + (i - n0)]) : 0;
        const float dx = exact_dist(tmem_row, Cl + (long long)k * p.r, p.r);
        if (have && (dx < bestx || (dx == bestx && k < bestk))) { bestx = dx; bestk = k; }
      }
      if (__any_sync(full, rescore && !balanced && !overflow && live)) {
        int e = 0, gid = 0;
        uint32_t mrem = 0;
        while (true) {
          while (mrem == 0 && e < n_ent) {
            if (entry_max(cl, e) >= thr) { mrem = entry_mask(cl, e, thr); gid = entry_gid(cl, e); }
            ++e;
          }
          const bool have = rescore && !balanced && !overflow && live && mrem != 0;
          if (!__any_sync(full, have)) break;
          int k = 0;
          if (have) { k = gid * 16 + __ffs(mrem) - 1; mrem &= mrem - 1; }
          const float dx = exact_dist(tmem_row, Cl + (long long)k * p.r, p.r);
#ifdef MAPL_DBG2
          if (lane == 0) atomicAdd(&g_dbg[blockIdx.x * 64 + 62], 1ull);
          if (have) atomicAdd(&g_dbg[blockIdx.x * 64 + 63], 1ull);
#endif
          if (have && (dx < bestx || (dx == bestx && k < bestk))) { bestx = dx; bestk = k; }
        }
      }
      // exhaustive pass over the codeword pieces a thread in overflow owns, done by its whole warp (below)
      for (unsigned owners = __ballot_sync(full, overflow); owners != 0; owners &= owners - 1) {
#ifdef MAPL_DBG2
        if (lane == 0) atomicAdd(&g_dbg[blockIdx.x * 64 + 58], 1ull);
        if (lane == __ffs(owners) - 1) { atomicAdd(&g_dbg[blockIdx.x * 64 + 57], hard ? 1ull : 0ull); atomicAdd(&g_dbg[blockIdx.x * 64 + 56], (unsigned long long)cl.novf); }
#endif
        exhaustive_half(tmem_row, Cl, p.r, p.K, h, lane, __ffs(owners) - 1, &bestx, &bestk);
      }
      if (warp == 2 && l == 1) { DBG(20) }
      xDist[mine] = bestx; xK[mine] = bestk;
      epi_sync();
#pragma unroll
      for (int hh = 0; hh < kParts; ++hh) {
        const float ox = xDist[hh * 128 + row];
        const int ok = xK[hh * 128 + row];
        if (ox < bestx || (ox == bestx && ok < bestk)) { bestx = ox; bestk = ok; }
      }
      if (bestk == 0x7fffffff) bestk = 0;       // dead rows
#pragma unroll
      for (int ll = 0; ll < 8; ++ll) if (ll == l) code_l[ll] = bestk;
      if (warp == 2 && l < 4) { DBG(6 + l * 4) }
      if (live && h == 0) p.codes[m * p.L + l] = bestk;
      if (l + 1 < p.L) {
        // rho -= C[l, k*] and, in the same pass, its fp16 operand for level l+1.  The scale only has to keep fp16 in
        // its normal range, so it comes from the bound max|rho_new| <= max|rho| + max|c| (no second pass for the exact
        // maximum); the exact ||rho_new||^2 and max|rho_new| are exchanged behind the hand-off.
        inv = inv_scale_of(amax + __ldg(lv + 4));
        float n2p, amaxp;
        // (staging buffers: the candidate lists' region is free until the next scan)
        rho_update(tmem_row, Cl, bestk, s.sRho, s.stash + (size_t)(warp - 2) * 32 * kStagePitch, row, p.r, h, lane,
                   live ? inv : 0.f, &n2p, &amaxp);
        xN2[mine] = n2p; xAmax[mine] = amaxp;
        write_ax(inv * __ldg(lv + 8 + 2), hard);
        if (warp == 2 && l == 1) { DBG(21) }
        publish_operand();
        epi_sync();
        n2 = 0.f; amax = 0.f;
#pragma unroll
        for (int hh = 0; hh < kParts; ++hh) { n2 += xN2[hh * 128 + row]; amax = fmaxf(amax, xAmax[hh * 128 + row]); }
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
                  int32_t* codes_out, cudaStream_t st, const int32_t* tok, const float* Tc, void* ovf_ws) {
  if (!tc_rvq_ok(d) || !pk.WBlo || !pk.Cb || !pk.hnb) return MAPL_ERR_UNSUPPORTED;
  RvqParams p;
  p.C = codebooks; p.lvl = pk.lvl; p.tok = tok; p.Tc = Tc;
  p.Zq = reinterpret_cast<__nv_bfloat16*>(Zq_out); p.codes = codes_out;
  p.N = d.n_tokens; p.d = d.d; p.r = d.r; p.L = d.rvq_levels; p.K = d.rvq_k;
  p.tile_m = tc_tile_m(d.n_tokens);
  p.ovf = reinterpret_cast<uint8_t*>(ovf_ws); p.kovf = kRvqOverflowEntries;
  p.nsplit = pk.WBlo2 ? 3 : 2;
  p.stage1_bytes = kTileBytes + p.nsplit * d.r * 64;
  // shared memory: four list entries (16-codeword groups) per thread -- the groups of one chunk take distinct FIFO
  // slots, and more entries only lengthen the pass over the lists after the scan (measured at config 2: 8 entries
  // 46.3 us, 4 entries 44.0 us, 5 spilled entries per launch) --, at least a chunk plus one codebook tile in flight,
  // and the rest of the level region for more ring tiles
  const int nkb = d.r / 64;
  const size_t cap = (size_t)227 * 1024 - 1024;
  p.kne = 0; p.ring_tiles = 0;
  for (int want = 2 * nkb; want >= nkb + 1 && p.kne == 0; --want) {
    p.kne = 4; p.ring_tiles = want; p.stages1 = 0;
    if (rvq_level_bytes(p) + rvq_tail_bytes(p.kne) > cap) p.kne = 0;
  }
  if (p.kne == 0) return MAPL_ERR_UNSUPPORTED;
  {   // the rest of the level region goes to the ring
    const size_t spare = cap - rvq_tail_bytes(p.kne) - rvq_level_bytes(p);
    p.ring_tiles += (int)(spare / kHalfTileBytes);
    if (p.ring_tiles > 16) p.ring_tiles = 16;
  }
  p.stages1 = (int)((cap - rvq_tail_bytes(p.kne)) / p.stage1_bytes);
  if (p.stages1 > 8) p.stages1 = 8;
  if (p.stages1 > d.d / 64) p.stages1 = d.d / 64;
  if (p.stages1 < 2) return MAPL_ERR_UNSUPPORTED;
  const size_t smem = 1024 + rvq_regionR(p) + rvq_tail_bytes(p.kne);
  if (smem > (size_t)227 * 1024) return MAPL_ERR_UNSUPPORTED;
  p.p1 = p.stages1 < kProducers ? p.stages1 : kProducers;
  p.p2 = p.ring_tiles / nkb < kProducers ? p.ring_tiles / nkb : kProducers;
  CUtensorMap tmH, tmWhi, tmWlo, tmWlo2, tmC, tmX;
  const uint64_t dd = (uint64_t)d.d, rr = (uint64_t)d.r, LK = (uint64_t)d.rvq_levels * d.rvq_k;
  if (!make_tmap_bf16_2d(&tmH, H, (uint64_t)d.n_tokens, dd, dd, 64, (uint32_t)p.tile_m)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmWhi, pk.WB, rr, dd, dd, 64, (uint32_t)d.r / 2)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmWlo, pk.WBlo, rr, dd, dd, 64, (uint32_t)d.r / 2)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmWlo2, pk.WBlo2 ? pk.WBlo2 : pk.WBlo, rr, dd, dd, 64, (uint32_t)d.r / 2)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmC, pk.Cb, LK, rr, rr, 64, kChunk / 2)) return MAPL_ERR_CUDA;
  if (!make_tmap_b16_k16_sw32(&tmX, pk.hnb, LK, kChunk / 2)) return MAPL_ERR_CUDA;
  MAPL_SMEM_OPT_IN(k_tc_encode_rvq, 227 * 1024);
  const unsigned tiles = ((unsigned)((d.n_tokens + p.tile_m - 1) / p.tile_m) + 1u) & ~1u;   // whole CTA pairs
  KernelScope ks(KID_TC_ENCODE_RVQ, st);
  MAPL_CUDA_CHECK(launch_pdl_pair(k_tc_encode_rvq, dim3(tiles), dim3(kThreads), smem, st, tmH, tmWhi, tmWlo, tmWlo2, tmC, tmX, p));
  return MAPL_OK;
}

}  // namespace mapl
