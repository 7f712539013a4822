// tc_stiefel.cu -- fp32-accurate GEMMs of the Stiefel step on the tensor cores (Eq. 4,
// PAPER.md:124 Eq. 7).
//
// tcgen05 has no fp32 kind, and one bf16 / TF32 pass cannot hold ||U^T U - I||_F <= 1e-5.  Every fp32
// operand x is therefore split EXACTLY into three bf16 planes x = x0 + x1 + x2 (x0 = bf16(x),
// x1 = bf16(x - x0), x2 = bf16(x - x0 - x1): 24 significant bits), and a product is the sum of the six
// plane pairs whose weight is above 2^-24:
//     a b  ~=  a0 b0 + a0 b1 + a1 b0 + a1 b1 + a0 b2 + a2 b0            (dropped: <= 2^-25 |a||b|)
// each pair exact in the tensor core (bf16 x bf16 -> fp32), accumulated in fp32 in TMEM.  Six MMAs per
// product still beat the FFMA pipes by a wide margin: the step's GEMMs are too small (<= 0.8 GFLOP)
// to fill those.
//
//   k_st_split   fp32 [rows, cols] -> bf16 planes [3][rows][cols] and/or transposed [3][cols][rows];
//                optionally applies the r x r maps of the step on the fly:
//                  mode 1  M  = (3 I - G) / 2                       (Newton-Schulz polynomial)
//                  mode 2  M1 = I + lr (S + S^T) / 2                (tangent projection + step, Eq. 4)
//                  mode 3  -(S + S^T) / 2                           (tangent projection alone: xi = G + U (-sym S))
//   k_tc_gemm3   C[M,N] (+)= sum_pairs A_i[M,K] B_j[N,K]^T, both K-major, 128 x 128 tile per CTA,
//                TMA-fed 2-stage ring of six [128 x 64] tiles; epilogue either C = acc + beta E (fp32
//                stores) or red.global.add (split over K).
// The tensor core adds into its fp32 accumulator with truncation, not round-to-nearest: a chain of ~100
// MMAs into one accumulator leaves a one-sided bias of ~2e-6 on the diagonal of X^T X, which the
// retraction inherits (measured: ||U^T U - I||_F 2.8e-5).  The k-blocks of a CTA therefore rotate over
// FOUR TMEM accumulators (24 MMAs each per visit) that the epilogue sums in registers with
// round-to-nearest; measured bias 7e-9, residual 2e-6, as the FFMA path.
#include <stdlib.h>

#include "profile.cuh"
#include "tc_common.cuh"
#include "tc_stiefel.cuh"
#include "tc_tile_ops.cuh"

namespace mapl {
namespace {
using namespace tc;

constexpr int kTile = 128 * 64 * 2;          // one [128 x 64] bf16 tile
constexpr int kStageBytes = 6 * kTile;       // three A planes + three B planes
constexpr int kStages = 2;

__device__ __forceinline__ void split3(float x, __nv_bfloat16* p0, __nv_bfloat16* p1, __nv_bfloat16* p2) {
  const __nv_bfloat16 a = __float2bfloat16_rn(x);
  const float r1 = x - __bfloat162float(a);
  const __nv_bfloat16 b = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(b);
  *p0 = a; *p1 = b; *p2 = __float2bfloat16_rn(r2);
}

// 32 x 32 tiles; blockIdx.y = batch item.  src [rows, cols] fp32; prow / ptr may be null.
// zero / nzero4: optional fp32 buffer (float4 count per batch item) cleared on the way (the next split-K target).
__global__ void __launch_bounds__(256) k_st_split(const float* __restrict__ src, int rows, int cols, int mode, float lr,
                                                  __nv_bfloat16* __restrict__ prow, __nv_bfloat16* __restrict__ ptr,
                                                  float4* __restrict__ zero, long long nzero4) {
  __shared__ float tile[32][33];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (zero != nullptr)
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < nzero4; i += (long long)gridDim.x * 256)
      zero[(long long)blockIdx.y * nzero4 + i] = make_float4(0.f, 0.f, 0.f, 0.f);
  const long long plane = (long long)rows * cols;
  src += (long long)blockIdx.y * plane;
  if (prow) prow += (long long)blockIdx.y * 3 * plane;
  if (ptr) ptr += (long long)blockIdx.y * 3 * plane;
  const int tiles_c = (cols + 31) / 32, tiles_r = (rows + 31) / 32;
  const int tx = threadIdx.x % 32, ty = threadIdx.x / 32;
  for (int t = blockIdx.x; t < tiles_c * tiles_r; t += gridDim.x) {
    const int r0 = (t / tiles_c) * 32, c0 = (t % tiles_c) * 32;
    for (int i = ty; i < 32; i += 8) {
      const int r = r0 + i, c = c0 + tx;
      float x = 0.f;
      if (r < rows && c < cols) {
        x = src[(long long)r * cols + c];
        if (mode == 1) x = 0.5f * ((r == c ? 3.f : 0.f) - x);
        if (mode == 2) x = (r == c ? 1.f : 0.f) + lr * 0.5f * (x + src[(long long)c * cols + r]);
        if (mode == 3) x = -0.5f * (x + src[(long long)c * cols + r]);
      }
      tile[i][tx] = x;
      if (prow && r < rows && c < cols) {
        __nv_bfloat16* o = prow + (long long)r * cols + c;
        split3(x, o, o + plane, o + 2 * plane);
      }
    }
    __syncthreads();
    if (ptr) {
      for (int i = ty; i < 32; i += 8) {
        const int c = c0 + i, r = r0 + tx;              // transposed element (c, r)
        if (c < cols && r < rows) {
          __nv_bfloat16* o = ptr + (long long)c * rows + r;
          split3(tile[tx][i], o, o + plane, o + 2 * plane);
        }
      }
    }
    __syncthreads();
  }
}

// Same for rows, cols multiples of 64 and modes 0 / 1, vectorised: 64 x 64 tiles, every thread converts 8 consecutive
// elements and stores 16 bytes per plane; the transposed planes go through shared memory so that 8 lanes write one
// whole 128-byte segment (the scalar kernel above writes 2 bytes per store instruction and lane).
__device__ __forceinline__ void split3x8(const float (&x)[8], __nv_bfloat16* o, long long plane) {
  uint32_t w[3][4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    __nv_bfloat16 a[2], b[2], c[2];
    split3(x[2 * j], &a[0], &b[0], &c[0]);
    split3(x[2 * j + 1], &a[1], &b[1], &c[1]);
    w[0][j] = (uint32_t)__bfloat16_as_ushort(a[0]) | ((uint32_t)__bfloat16_as_ushort(a[1]) << 16);
    w[1][j] = (uint32_t)__bfloat16_as_ushort(b[0]) | ((uint32_t)__bfloat16_as_ushort(b[1]) << 16);
    w[2][j] = (uint32_t)__bfloat16_as_ushort(c[0]) | ((uint32_t)__bfloat16_as_ushort(c[1]) << 16);
  }
#pragma unroll
  for (int pl = 0; pl < 3; ++pl) *reinterpret_cast<uint4*>(o + pl * plane) = make_uint4(w[pl][0], w[pl][1], w[pl][2], w[pl][3]);
}

__global__ void __launch_bounds__(256) k_st_split64(const float* __restrict__ src, int rows, int cols, int mode,
                                                    __nv_bfloat16* __restrict__ prow, __nv_bfloat16* __restrict__ ptr,
                                                    float4* __restrict__ zero, long long nzero4) {
  __shared__ float tile[64][65];
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (zero != nullptr)
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < nzero4; i += (long long)gridDim.x * 256)
      zero[(long long)blockIdx.y * nzero4 + i] = make_float4(0.f, 0.f, 0.f, 0.f);
  const long long plane = (long long)rows * cols;
  src += (long long)blockIdx.y * plane;
  if (prow) prow += (long long)blockIdx.y * 3 * plane;
  if (ptr) ptr += (long long)blockIdx.y * 3 * plane;
  const int tiles_c = cols / 64, tiles_r = rows / 64, t = threadIdx.x;
  for (int tl = blockIdx.x; tl < tiles_c * tiles_r; tl += gridDim.x) {
    const int r0 = (tl / tiles_c) * 64, c0 = (tl % tiles_c) * 64;
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int idx = t + 256 * u, i = idx / 8, c8 = (idx % 8) * 8;         // row i of the tile, columns c8 .. c8+7
      const int r = r0 + i, c = c0 + c8;
      const float4 lo = *reinterpret_cast<const float4*>(src + (long long)r * cols + c);
      const float4 hi = *reinterpret_cast<const float4*>(src + (long long)r * cols + c + 4);
      float x[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
      if (mode == 1) {
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 0.5f * ((r == c + j ? 3.f : 0.f) - x[j]);
      }
      if (ptr) {
#pragma unroll
        for (int j = 0; j < 8; ++j) tile[i][c8 + j] = x[j];
      }
      if (prow) split3x8(x, prow + (long long)r * cols + c, plane);
    }
    if (ptr) {
      __syncthreads();
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int idx = t + 256 * u, cc = idx / 8, r8 = (idx % 8) * 8;      // transposed row cc, elements r8 .. r8+7
        float x[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = tile[r8 + j][cc];
        split3x8(x, ptr + (long long)(c0 + cc) * rows + r0 + r8, plane);
      }
      __syncthreads();
    }
  }
}

struct Gemm3Params {
  float* C; const float* E;
  float beta;
  int M, N, K;              // per batch item; M, N multiples of 128, K multiple of 64
  int kb_per_split;         // k-blocks (of 64) per blockIdx.z split
  int nsplit;               // blockIdx.z = batch * nsplit + split
  int atomic;
  long long sC;             // batch stride of C / E (elements)
};

__global__ void __launch_bounds__(192, 1)
k_tc_gemm3(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const Gemm3Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)kStages * kStageBytes);
  uint64_t* empty = full + kStages;
  uint64_t* acc_full = empty + kStages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_full + 1);

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int b = blockIdx.z / p.nsplit, split = blockIdx.z % p.nsplit;
  const int m0 = blockIdx.x * 128, n0 = blockIdx.y * 128;
  const int nkb_all = p.K / 64;
  const int kb0 = split * p.kb_per_split, kb1 = min(nkb_all, kb0 + p.kb_per_split);
  const int nkb = kb1 > kb0 ? kb1 - kb0 : 0;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmA); tma_prefetch_desc(&tmB);
    for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_init(acc_full, 1);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<512>(tmem_slot);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_d = *tmem_slot;
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");

  if (nkb > 0) {
    if (warp == 0) {
      if (elect_one()) {
        for (int it = 0; it < nkb; ++it) {
          const int s = it % kStages, kc = (kb0 + it) * 64;
          mbar_wait(&empty[s], ((it / kStages) & 1) ^ 1);
          mbar_arrive_expect_tx(&full[s], kStageBytes);
          uint8_t* a = smem + (size_t)s * kStageBytes;
#pragma unroll
          for (int pl = 0; pl < 3; ++pl) {
            tma_load_2d(a + pl * kTile, &tmA, &full[s], kc, (b * 3 + pl) * p.M + m0, kEvictLast);
            tma_load_2d(a + (3 + pl) * kTile, &tmB, &full[s], kc, (b * 3 + pl) * p.N + n0, kEvictLast);
          }
        }
      }
    } else if (warp == 1) {
      if (elect_one()) {
        const uint32_t idesc = make_idesc_bf16(128, 128, false, false);
        // plane pairs (A plane, B plane), smallest weights first
        const int pa[6] = {2, 0, 1, 1, 0, 0}, pb[6] = {0, 2, 1, 0, 1, 0};
        for (int it = 0; it < nkb; ++it) {
          const int s = it % kStages;
          mbar_wait(&full[s], (it / kStages) & 1);
          tc_fence_after_sync();
          const uint32_t base = smem_u32(smem + (size_t)s * kStageBytes);
#pragma unroll
          for (int q = 0; q < 6; ++q) {
            const uint32_t a = base + pa[q] * kTile, bb = base + (3 + pb[q]) * kTile;
#pragma unroll
            for (int k = 0; k < 4; ++k)
              umma_bf16(tmem_d + (it & 3) * 128, desc_kmajor_sw128(a + k * 32), desc_kmajor_sw128(bb + k * 32), idesc,
                        (it >= 4) || (q | k) != 0);
          }
          umma_commit(&empty[s]);
        }
        umma_commit(acc_full);
      }
    } else {
      const int q = warp & 3, row = q * 32 + lane;
      const long long off = (long long)b * p.sC + (long long)(m0 + row) * p.N + n0;
      float* dst = p.C + off;
      mbar_wait(acc_full, 0);
      tc_fence_after_sync();
      const int nacc = nkb < 4 ? nkb : 4;
      for (int cc = 0; cc < 4; ++cc) {
        uint32_t v[32];
        tmem_ld32(tmem_d + ((uint32_t)(q * 32) << 16) + cc * 32, v);
        tmem_ld_wait();
        for (int a = 1; a < nacc; ++a) {             // the other accumulators, summed round-to-nearest
          uint32_t w[32];
          tmem_ld32(tmem_d + ((uint32_t)(q * 32) << 16) + a * 128 + cc * 32, w);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) + __uint_as_float(w[i]));
        }
        if (p.atomic) {
#pragma unroll
          for (int i = 0; i < 8; ++i)
            asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + cc * 32 + i * 4),
                         "f"(__uint_as_float(v[4 * i])), "f"(__uint_as_float(v[4 * i + 1])), "f"(__uint_as_float(v[4 * i + 2])),
                         "f"(__uint_as_float(v[4 * i + 3])) : "memory");
        } else {
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            float4 o = make_float4(__uint_as_float(v[4 * i]), __uint_as_float(v[4 * i + 1]), __uint_as_float(v[4 * i + 2]),
                                   __uint_as_float(v[4 * i + 3]));
            if (p.E) {
              const float4 e = __ldg(reinterpret_cast<const float4*>(p.E + off + cc * 32 + i * 4));
              o.x = fmaf(p.beta, e.x, o.x); o.y = fmaf(p.beta, e.y, o.y); o.z = fmaf(p.beta, e.z, o.z); o.w = fmaf(p.beta, e.w, o.w);
            }
            *reinterpret_cast<float4*>(dst + cc * 32 + i * 4) = o;
          }
        }
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after_sync();
    tmem_dealloc<512>(tmem_d);
  }
}

}  // namespace

// r = 128 was measured slower on this path (158 vs 125 us for 3 projectors): the FFMA kernels keep it
bool tc_st_ok(int d, int r) { return d % 128 == 0 && r % 128 == 0 && r >= 256 && r <= 1024; }

size_t tc_st_plane_bytes(int d, int r, int batch) {   // one set of planes of a [d,r] matrix
  return align_up((size_t)batch * 3 * d * r * 2, 256);
}

int tc_st_split(const float* src, int rows, int cols, int batch, int mode, float lr, __nv_bfloat16* prow,
                __nv_bfloat16* ptr, cudaStream_t st, float* zero, long long nzero) {
  KernelScope ks(KID_ST_SPLIT, st);
  if (mode <= 1 && rows % 64 == 0 && cols % 64 == 0) {
    const int tiles64 = (rows / 64) * (cols / 64);
    MAPL_CUDA_CHECK(tc::launch_pdl(k_st_split64, dim3(tiles64 < 1024 ? tiles64 : 1024, batch), dim3(256), 0, st, src, rows, cols, mode,
                                   prow, ptr, reinterpret_cast<float4*>(zero), nzero / 4));
    return MAPL_OK;
  }
  const int tiles = ((rows + 31) / 32) * ((cols + 31) / 32);
  MAPL_CUDA_CHECK(tc::launch_pdl(k_st_split, dim3(tiles < 1024 ? tiles : 1024, batch), dim3(256), 0, st, src, rows, cols, mode, lr,
                                 prow, ptr, reinterpret_cast<float4*>(zero), nzero / 4));
  return MAPL_OK;
}

// C[b] (+)= A[b] B[b]^T from planes Ap [batch][3][M][K], Bp [batch][3][N][K].  nsplit > 1: C must be zeroed,
// the K range is split and partial sums are added with red.global.add.  Else C = acc + beta E.
int tc_st_gemm3(const __nv_bfloat16* Ap, const __nv_bfloat16* Bp, int M, int N, int K, int batch, float* C, const float* E,
                float beta, int nsplit, cudaStream_t st) {
  if (M % 128 || N % 128 || K % 64) return MAPL_ERR_UNSUPPORTED;
  CUtensorMap tmA, tmB;
  if (!make_tmap_bf16_2d(&tmA, Ap, (uint64_t)batch * 3 * M, (uint64_t)K, (uint64_t)K, 64, 128)) return MAPL_ERR_CUDA;
  if (!make_tmap_bf16_2d(&tmB, Bp, (uint64_t)batch * 3 * N, (uint64_t)K, (uint64_t)K, 64, 128)) return MAPL_ERR_CUDA;
  Gemm3Params p;
  p.C = C; p.E = E; p.beta = beta; p.M = M; p.N = N; p.K = K;
  const int nkb = K / 64;
  if (nsplit < 1) nsplit = 1;
  if (nsplit > nkb) nsplit = nkb;
  p.kb_per_split = (nkb + nsplit - 1) / nsplit;
  p.nsplit = (nkb + p.kb_per_split - 1) / p.kb_per_split;
  p.atomic = p.nsplit > 1 ? 1 : 0;
  p.sC = (long long)M * N;
  const size_t smem = (size_t)kStages * kStageBytes + 1024 + 256;
  MAPL_SMEM_OPT_IN(k_tc_gemm3, 227 * 1024);
  KernelScope ks(KID_ST_GEMM3, st);
  MAPL_CUDA_CHECK(tc::launch_pdl(k_tc_gemm3, dim3(M / 128, N / 128, batch * p.nsplit), dim3(192), smem, st, tmA, tmB, p));
  return MAPL_OK;
}

}  // namespace mapl
