// tc_codec.cu -- envelope checks and the parameter pack shared by the tcgen05 codec kernels
// (tc_encode.cu, tc_encode_rvq.cu, tc_decode.cu, tc_backward.cu).
#include "tc_codec.cuh"

#include <cuda_fp16.h>
#include <stdlib.h>

#include "profile.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {

bool tc_shape_ok(const mapl_boundary_desc& d) {
  if (d.act_dtype != MAPL_BF16) return false;
  if (d.d % 256 != 0 || d.d < 256) return false;      // the decode / dH chunk pipeline works in 256-column chunks
  if (d.r != 64 && d.r != 128 && d.r != 256) return false;
  if (d.anchor_rank != 0 && d.anchor_rank != 64 && d.anchor_rank != 128) return false;
  if (d.n_tokens < 1) return false;
  return true;
}

bool tc_rvq_ok(const mapl_boundary_desc& d) {
  return tc_shape_ok(d) && d.rvq_levels > 0 && d.rvq_k >= 128 && d.rvq_k % 128 == 0 && d.rvq_k <= 8192;
}

TcPack tc_pack_layout(const mapl_boundary_desc& d, char* base) {
  TcPack p;
  if (!tc_shape_ok(d)) return p;
  size_t off = 0;
  auto seg = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return base ? base + o : nullptr; };
  p.kc = d.r + d.anchor_rank;
  p.WB = reinterpret_cast<__nv_bfloat16*>(seg((size_t)p.kc * d.d * 2));
  p.Wd = reinterpret_cast<__nv_bfloat16*>(seg((size_t)p.kc * d.d * 2));
  if (d.rvq_levels > 0) {
    const size_t LK = (size_t)d.rvq_levels * d.rvq_k;
    p.WBlo = reinterpret_cast<__nv_bfloat16*>(seg((size_t)d.r * d.d * 2));
    if (d.rvq_levels >= 3) p.WBlo2 = reinterpret_cast<__nv_bfloat16*>(seg((size_t)d.r * d.d * 2));
    p.Cb = reinterpret_cast<__nv_bfloat16*>(seg(LK * d.r * 2));
    p.hnb = reinterpret_cast<__nv_bfloat16*>(seg(LK * 16 * 2));
    p.hn = reinterpret_cast<float*>(seg(LK * 4));
    p.rowamax = reinterpret_cast<float*>(seg(LK * 4));
    p.lvl = reinterpret_cast<float*>(seg(8 * 8 * 4));
  }
  p.bytes = off;
  return p;
}

size_t tc_scratch_bytes(const mapl_boundary_desc& d) {
  if (!tc_shape_ok(d)) return 0;
  return d.rvq_levels > 0 ? align_up((size_t)d.n_tokens * d.r * 2, 256) : 0;
}

size_t tc_rvq_overflow_bytes(const mapl_boundary_desc& d) {
  if (!tc_rvq_ok(d)) return 0;
  const long long tm = tc_tile_m(d.n_tokens);
  const long long tiles = ((d.n_tokens + tm - 1) / tm + 1) & ~1ll;
  return (size_t)tiles * 256 * kRvqOverflowEntries * kRvqOverflowBytes;
}

int tc_tile_m(long long N) {
  const long long per_wave = 148ll * 128;
  const long long waves = (N + per_wave - 1) / per_wave;
  long long t = (N + 148 * waves - 1) / (148 * waves);
  t = (t + 7) / 8 * 8;
  if (t > 128) t = 128;
  if (t < 8) t = 8;
  return (int)t;
}

int tc_tile_m4(long long N) {
  const long long ctas = 132, per_wave = ctas * 128;
  const long long waves = (N + per_wave - 1) / per_wave;
  long long t = (N + ctas * waves - 1) / (ctas * waves);
  t = (t + 7) / 8 * 8;
  if (t > 128) t = 128;
  if (t < 8) t = 8;
  return (int)t;
}

int tc_pairs_per_cluster() {
  static const int nq = (getenv("MAPL_NQ") && getenv("MAPL_NQ")[0] == '2') ? 2 : 1;
  return nq;
}

namespace {

struct PackJob {
  const float* src; int rows, cols;        // src is [rows, cols] fp32 row-major
  __nv_bfloat16* dst; long long pitch;     // dst element (i,j) -> dst[i*pitch + j] (after optional transpose)
  int transpose;
  int mode;                                // 0: bf16(x)   1: bf16(x - float(bf16(x))), the second split term
                                           // 2: fp16(x * scale[8 * (src_row / rows_per_scale) + 3])  (16-bit store)
                                           // 3: the third split term bf16(x - hi - lo)
  const float* scale; int rows_per_scale;
};
struct PackArgs { PackJob job[7]; int njobs; };

__device__ __forceinline__ __nv_bfloat16 pack_term(float x, int mode, float sc) {
  if (mode == 2) {
    const unsigned short h = __half_as_ushort(__float2half_rn(x * sc));
    return *reinterpret_cast<const __nv_bfloat16*>(&h);
  }
  const __nv_bfloat16 hi = __float2bfloat16_rn(x);
  if (mode == 0) return hi;
  const float r1 = x - __bfloat162float(hi);          // exact
  const __nv_bfloat16 lo = __float2bfloat16_rn(r1);
  return mode == 1 ? lo : __float2bfloat16_rn(r1 - __bfloat162float(lo));
}

// 64 x 64 tiles (every dimension of a pack job is a multiple of 64 inside the tensor-core envelope); blockIdx.y = job.
// 16-byte loads, 8-byte stores (four 16-bit values), the transposition through shared memory.  Programmatic dependent
// launch: the next kernel's prologue may start at once, and the sources are read only after the kernels before this one
// have completed (U may just have been written by the Stiefel step).
__global__ void __launch_bounds__(256) k_tc_pack(const PackArgs a) {
  __shared__ float tile[64][65];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const PackJob j = a.job[blockIdx.y];
  const int tiles_c = j.cols / 64, tiles_r = j.rows / 64;
  const int q = threadIdx.x % 16, y = threadIdx.x / 16;       // q: group of 4 consecutive elements, y: 0 .. 15
  for (int t = blockIdx.x; t < tiles_c * tiles_r; t += gridDim.x) {
    const int r0 = (t / tiles_c) * 64, c0 = (t % tiles_c) * 64;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int r = y + 16 * i;
      const float4 x = *reinterpret_cast<const float4*>(j.src + (long long)(r0 + r) * j.cols + c0 + 4 * q);
      tile[r][4 * q + 0] = x.x; tile[r][4 * q + 1] = x.y; tile[r][4 * q + 2] = x.z; tile[r][4 * q + 3] = x.w;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int u = y + 16 * i;                                // dst row inside the tile
      __nv_bfloat16 o[4];
      if (j.transpose) {                                       // dst[c0 + u][r0 + 4 q ..] = src[r0 + 4 q ..][c0 + u]
#pragma unroll
        for (int e = 0; e < 4; ++e) o[e] = pack_term(tile[4 * q + e][u], j.mode, 1.f);
        *reinterpret_cast<uint2*>(j.dst + (long long)(c0 + u) * j.pitch + r0 + 4 * q) = *reinterpret_cast<const uint2*>(o);
      } else {
        const float sc = j.mode == 2 ? j.scale[8 * ((r0 + u) / j.rows_per_scale) + 3] : 1.f;
#pragma unroll
        for (int e = 0; e < 4; ++e) o[e] = pack_term(tile[u][4 * q + e], j.mode, sc);
        *reinterpret_cast<uint2*>(j.dst + (long long)(r0 + u) * j.pitch + c0 + 4 * q) = *reinterpret_cast<const uint2*>(o);
      }
    }
    __syncthreads();
  }
}

// one warp per codeword row: hn = 0.5 ||c||^2, rowamax = max_j |c_j|
__global__ void __launch_bounds__(256) k_tc_cb_stats(const float* __restrict__ C, float* __restrict__ hn,
                                                     float* __restrict__ rowamax, int rows, int r) {
  const int row = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
  if (row >= rows) return;
  float s = 0.f, m = 0.f;
  for (int j = lane; j < r; j += 32) { const float c = C[(long long)row * r + j]; s = fmaf(c, c, s); m = fmaxf(m, fabsf(c)); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o)); }
  if (lane == 0) { hn[row] = 0.5f * s; rowamax[row] = m; }
}

// one block per level: lvl[8 l + ...] = {cmax sc, qmax, 2^g, sc, 2^e, cmax}: sc = 2^-e with max|c| * sc in [0.5, 1)
// (powers of two: the fp16 codebook copy C * sc is exact up to the fp16 rounding), cmax = max_k ||c_k||,
// q_k = hn_k sc 2^-g with g >= 0 the smallest integer that brings max_k q_k to <= 2^15 (fp16 range)
__global__ void __launch_bounds__(256) k_tc_cmax(const float* __restrict__ hn, const float* __restrict__ rowamax,
                                                 float* __restrict__ lvl, int K) {
  __shared__ float red[8], red2[8];
  float m = 0.f, a = 0.f;
  for (int k = threadIdx.x; k < K; k += 256) {
    m = fmaxf(m, hn[(long long)blockIdx.x * K + k]);
    a = fmaxf(a, rowamax[(long long)blockIdx.x * K + k]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o)); a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, o)); }
  if (threadIdx.x % 32 == 0) { red[threadIdx.x / 32] = m; red2[threadIdx.x / 32] = a; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < 8; ++i) { m = fmaxf(m, red[i]); a = fmaxf(a, red2[i]); }
    const float cmax = sqrtf(2.f * m);
    int eb = (int)((__float_as_uint(a) >> 23) & 0xffu);
    eb = eb < 2 ? 126 : (eb > 250 ? 250 : eb);             // all-zero / denormal codebook: scale 1
    const float sc = __uint_as_float((uint32_t)(253 - eb) << 23);
    float q = m * sc, pg = 1.f;
    while (q > 32768.f && pg < 1e30f) { q *= 0.5f; pg *= 2.f; }
    float* o = lvl + 8 * blockIdx.x;
    o[0] = cmax * sc; o[1] = q; o[2] = pg; o[3] = sc; o[4] = __uint_as_float((uint32_t)(eb + 1) << 23); o[5] = cmax;
    o[6] = 0.f; o[7] = 0.f;
  }
}

// hnb[row, 0..2] = -(fp16 three-term split of q = hn[row] sc / 2^g), hnb[row, 3..15] = 0.  The split is exact up to
// 2^-33 q + 2^-25 (each remainder is exact in fp32; the last one is dropped).
__global__ void __launch_bounds__(256) k_tc_hnb(const float* __restrict__ hn, const float* __restrict__ lvl,
                                                __nv_bfloat16* __restrict__ hnb, int rows, int K) {
  const int row = blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= rows) return;
  const float* o = lvl + 8 * (row / K);
  float q = hn[row] * o[3] / o[2];
  unsigned short h[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) h[i] = 0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const __half p = __float2half_rn(q);
    q -= __half2float(p);
    h[i] = __half_as_ushort(__float2half_rn(-__half2float(p)));
  }
  uint4* dst = reinterpret_cast<uint4*>(hnb + (long long)row * 16);
  dst[0] = make_uint4(h[0] | ((uint32_t)h[1] << 16), h[2] | ((uint32_t)h[3] << 16), 0u, 0u);
  dst[1] = make_uint4(0u, 0u, 0u, 0u);
}

}  // namespace

int tc_pack_build(const mapl_boundary_desc& d, const float* U, const float* B, const float* codebooks,
                  const TcPack& p, cudaStream_t st) {
  const bool rvq = d.rvq_levels > 0 && p.hn && codebooks;
  if (rvq) {
    const int rows = d.rvq_levels * d.rvq_k;
    {
      KernelScope ks(KID_TC_PACK, st);
      k_tc_cb_stats<<<(rows + 7) / 8, 256, 0, st>>>(codebooks, p.hn, p.rowamax, rows, d.r);
      MAPL_CUDA_CHECK(cudaGetLastError());
    }
    {
      KernelScope ks(KID_TC_PACK, st);
      k_tc_cmax<<<d.rvq_levels, 256, 0, st>>>(p.hn, p.rowamax, p.lvl, d.rvq_k);
      MAPL_CUDA_CHECK(cudaGetLastError());
    }
    KernelScope ks(KID_TC_PACK, st);
    k_tc_hnb<<<(rows + 255) / 256, 256, 0, st>>>(p.hn, p.lvl, p.hnb, rows, d.rvq_k);
    MAPL_CUDA_CHECK(cudaGetLastError());
  }
  PackArgs a;
  a.njobs = 0;
  const int ra = d.anchor_rank;
  a.job[a.njobs++] = PackJob{U, d.d, d.r, p.WB, d.d, 1, 0, nullptr, 1};                            // WB[j][i] = U[i][j]
  a.job[a.njobs++] = PackJob{U, d.d, d.r, p.Wd, p.kc, 0, 0, nullptr, 1};                           // Wd[i][j] = U[i][j]
  if (ra && B) {
    a.job[a.njobs++] = PackJob{B, ra, d.d, p.WB + (long long)d.r * d.d, d.d, 0, 0, nullptr, 1};
    a.job[a.njobs++] = PackJob{B, ra, d.d, p.Wd + d.r, p.kc, 1, 0, nullptr, 1};                    // Wd[i][r+q] = B[q][i]
  }
  if (d.rvq_levels > 0 && p.WBlo) {
    a.job[a.njobs++] = PackJob{U, d.d, d.r, p.WBlo, d.d, 1, 1, nullptr, 1};
    if (p.WBlo2) a.job[a.njobs++] = PackJob{U, d.d, d.r, p.WBlo2, d.d, 1, 3, nullptr, 1};
    if (rvq) a.job[a.njobs++] = PackJob{codebooks, d.rvq_levels * d.rvq_k, d.r, p.Cb, d.r, 0, 2, p.lvl, d.rvq_k};
  }
  {
    KernelScope ks(KID_TC_PACK, st);
    int max_tiles = 1;
    for (int i = 0; i < a.njobs; ++i) {
      if (a.job[i].rows % 64 || a.job[i].cols % 64) return MAPL_ERR_UNSUPPORTED;     // cannot happen inside the envelope
      const int t = (a.job[i].rows / 64) * (a.job[i].cols / 64);
      if (t > max_tiles) max_tiles = t;
    }
    // blocks beyond a job's tile count exit at once
    MAPL_CUDA_CHECK(tc::launch_pdl(k_tc_pack, dim3(max_tiles < 592 ? max_tiles : 592, a.njobs), dim3(256), 0, st, a));
  }
  return MAPL_OK;
}

}  // namespace mapl
