// simt_codec.cu -- general-shape fp32 kernels of the codec: fused projection + residual VQ
// (z stays in shared memory between levels), dequantisation, anchor-gradient scatter.
#include <float.h>

#include "common.cuh"
#include "profile.cuh"

namespace mapl {
namespace {

constexpr int TOK = 64, CW = 64, BK = 16, NT = 256, PAD = 4, LD = TOK + PAD;
constexpr int MAXL = 8;

// ---------------------------------------------------------------- 0.5*||c||^2 per codeword
__global__ void k_half_sqnorm(const float* __restrict__ C, float* __restrict__ out, int rows, int r) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) / 32, lane = threadIdx.x % 32;
  if (warp >= rows) return;
  float s = 0.f;
  for (int j = lane; j < r; j += 32) { float c = C[(long long)warp * r + j]; s = fmaf(c, c, s); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) out[warp] = 0.5f * s;
}

// ---------------------------------------------------------------- fused project + RVQ
// One CTA = 64 tokens.  rhoT[k][t] (k < r) holds the residual, transposed so the 4x4 micro-kernel
// reads it like an A tile.  Per level the codebook streams through Bs in 64-codeword tiles;
// score_k = 0.5||c_k||^2 - rho.c_k, argmin with lowest index on ties (S4).
template <bool kActBf16>
__global__ void __launch_bounds__(NT) k_simt_encode_rvq(
    const void* __restrict__ Hv, const float* __restrict__ U, const float* __restrict__ C,
    const float* __restrict__ half_norm, void* __restrict__ Zq, int32_t* __restrict__ codes,
    long long N, int d, int r, int L, int K, const int32_t* __restrict__ tok, const float* __restrict__ Tc) {
  extern __shared__ __align__(16) float smem[];
  const int rpad = (r + BK - 1) / BK * BK;
  float(*rhoT)[LD] = reinterpret_cast<float(*)[LD]>(smem);                 // [rpad][LD]
  float(*As)[LD] = reinterpret_cast<float(*)[LD]>(smem + (size_t)rpad * LD);  // [BK][LD]
  float(*Bs)[LD] = As + BK;                                                // [BK][LD]
  int* code_s = reinterpret_cast<int*>(Bs + BK);                           // [TOK][MAXL]

  const int t = threadIdx.x, tx = t % 16, ty = t / 16;
  const long long m0 = (long long)blockIdx.x * TOK;

  for (int i = t; i < rpad * LD; i += NT) smem[i] = 0.f;
  __syncthreads();

  // ---- phase 0: rhoT = (H tile . U)^T
  for (int n0 = 0; n0 < r; n0 += CW) {
    float acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
    for (int k0 = 0; k0 < d; k0 += BK) {
#pragma unroll
      for (int it = 0; it < (TOK * BK) / NT; ++it) {   // H tile: k contiguous
        int idx = t + it * NT, k = idx % BK, i = idx / BK;
        long long m = m0 + i;
        float v = 0.f;
        if (m < N && k0 + k < d) {
          long long gi = m * d + k0 + k;
          v = kActBf16 ? __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(Hv)[gi])
                       : reinterpret_cast<const float*>(Hv)[gi];
        }
        As[k][i] = v;
      }
#pragma unroll
      for (int it = 0; it < (CW * BK) / NT; ++it) {    // U tile: n contiguous
        int idx = t + it * NT, n = idx % CW, k = idx / CW;
        float v = 0.f;
        if (n0 + n < r && k0 + k < d) v = U[(long long)(k0 + k) * r + n0 + n];
        Bs[k][n] = v;
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < BK; ++k) {
        const float4 a = *reinterpret_cast<const float4*>(&As[k][ty * 4]);
        const float4 b = *reinterpret_cast<const float4*>(&Bs[k][tx * 4]);
        const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
      }
      __syncthreads();
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int n = n0 + tx * 4 + j;
      if (n < r)
#pragma unroll
        for (int i = 0; i < 4; ++i) rhoT[n][ty * 4 + i] = acc[i][j];
    }
  }
  __syncthreads();
  if (Tc != nullptr) {   // sender-side centring (Eq. 1): z -= T[tok], T = A_s (B_s U) per vocabulary entry
    for (int i = t; i < r * TOK; i += NT) {
      const int k = i % r, tt = i / r;
      const long long m = m0 + tt;
      if (m < N) rhoT[k][tt] -= Tc[(long long)tok[m] * r + k];
    }
    __syncthreads();
  }

  // ---- levels
  for (int l = 0; l < L; ++l) {
    const float* Cl = C + (long long)l * K * r;
    const float* hn = half_norm + (long long)l * K;
    float best[4] = {FLT_MAX, FLT_MAX, FLT_MAX, FLT_MAX};
    int bidx[4] = {0, 0, 0, 0};
    for (int c0 = 0; c0 < K; c0 += CW) {
      float acc[4][4];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
      for (int k0 = 0; k0 < r; k0 += BK) {
#pragma unroll
        for (int it = 0; it < (CW * BK) / NT; ++it) {  // codebook tile: k contiguous
          int idx = t + it * NT, k = idx % BK, n = idx / BK;
          float v = 0.f;
          if (c0 + n < K && k0 + k < r) v = Cl[(long long)(c0 + n) * r + k0 + k];
          Bs[k][n] = v;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < BK; ++k) {
          const float4 a = *reinterpret_cast<const float4*>(&rhoT[k0 + k][ty * 4]);
          const float4 b = *reinterpret_cast<const float4*>(&Bs[k][tx * 4]);
          const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
          for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
        }
        __syncthreads();
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int n = c0 + tx * 4 + j;
        if (n < K) {
          const float h = hn[n];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float s = h - acc[i][j];
            if (s < best[i]) { best[i] = s; bidx[i] = n; }   // n increases: ties keep the lowest
          }
        }
      }
    }
    // combine the 16 lanes (tx) that share a token row: lexicographic (score, index)
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) {
        const float os = __shfl_xor_sync(0xffffffffu, best[i], o);
        const int oi = __shfl_xor_sync(0xffffffffu, bidx[i], o);
        if (os < best[i] || (os == best[i] && oi < bidx[i])) { best[i] = os; bidx[i] = oi; }
      }
      if (tx == 0) {
        code_s[(ty * 4 + i) * MAXL + l] = bidx[i];
        const long long m = m0 + ty * 4 + i;
        if (m < N) codes[m * L + l] = bidx[i];
      }
    }
    __syncthreads();
    for (int idx = t; idx < TOK * r; idx += NT) {          // rho <- rho - C[l, code, :]
      const int j = idx % r, tk = idx / r;
      rhoT[j][tk] -= Cl[(long long)code_s[tk * MAXL + l] * r + j];
    }
    __syncthreads();
  }

  if (Zq != nullptr) {                                     // zhat = sum_l C[l, code_l, :]
    for (int idx = t; idx < TOK * r; idx += NT) {
      const int j = idx % r, tk = idx / r;
      const long long m = m0 + tk;
      if (m >= N) continue;
      float s = 0.f;
      for (int l = 0; l < L; ++l) s += C[((long long)l * K + code_s[tk * MAXL + l]) * r + j];
      if (kActBf16) reinterpret_cast<__nv_bfloat16*>(Zq)[m * r + j] = __float2bfloat16_rn(s);
      else reinterpret_cast<float*>(Zq)[m * r + j] = s;
    }
  }
}

__global__ void k_dequant(const int32_t* __restrict__ codes, const float* __restrict__ C,
                          float* __restrict__ Zhat, long long N, int r, int L, int K) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * r) return;
  const long long n = idx / r;
  const int j = (int)(idx % r);
  float s = 0.f;
  for (int l = 0; l < L; ++l) s += C[((long long)l * K + codes[n * L + l]) * r + j];
  Zhat[idx] = s;
}

// dA[tok_n, :] += gA[n, :].  Token ids are skewed (Zipf: the hottest id owns ~14 % of the rows), so one atomic per row
// element serialises in L2 on the hot rows.  Per block of 128 tokens: rank the ids (counting sort in shared memory),
// then every run of equal ids is summed by ra / 4 threads (one float4 column chunk each, rows read once from L2) and
// leaves the block as ONE red per distinct id and chunk.  ra % 4 == 0; other widths take the element-wise path.
__global__ void __launch_bounds__(128) k_scatter_add_rows(const float* __restrict__ gA, const int32_t* __restrict__ tok,
                                                          float* __restrict__ dA, long long N, int ra) {
  __shared__ int sTok[128], sSorted[128], sOrder[128];
  const int t = threadIdx.x, nv = ra / 4;
  for (long long base = (long long)blockIdx.x * 128; base < N; base += (long long)gridDim.x * 128) {
    const int cnt = (int)(N - base < 128 ? N - base : 128);
    const int my = t < cnt ? tok[base + t] : 0x7fffffff;
    sTok[t] = my;
    __syncthreads();
    int rank = 0;
#pragma unroll 8
    for (int j = 0; j < 128; ++j) {
      const int o = sTok[j];
      rank += (o < my || (o == my && j < t)) ? 1 : 0;
    }
    sSorted[rank] = my;
    sOrder[rank] = t;
    __syncthreads();
    // work items: (sorted position, column chunk); a thread that lands on the head of a run sums the run
    for (int item = t; item < cnt * nv; item += 128) {
      const int pos = item / nv, cc = item - pos * nv;
      const int id = sSorted[pos];
      if (pos > 0 && sSorted[pos - 1] == id) continue;
      float4 acc = __ldg(reinterpret_cast<const float4*>(gA + (base + sOrder[pos]) * ra) + cc);
      for (int q = pos + 1; q < cnt && sSorted[q] == id; ++q) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(gA + (base + sOrder[q]) * ra) + cc);
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
      }
      float* dst = dA + (long long)id * ra + cc * 4;
      asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(acc.x), "f"(acc.y), "f"(acc.z), "f"(acc.w) : "memory");
    }
    __syncthreads();
  }
}

__global__ void k_scatter_add_elems(const float* __restrict__ gA, const int32_t* __restrict__ tok,
                                    float* __restrict__ dA, long long N, int ra) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * ra) return;
  const long long n = idx / ra;
  const int q = (int)(idx % ra);
  atomicAdd(dA + (long long)tok[n] * ra + q, gA[idx]);
}

}  // namespace

// D[tok_n, :] += X[n, :]: one warp per token row, fp32 atomics (reds)
template <bool kBf16>
__global__ void k_scatter_act_rows(const void* __restrict__ Xv, const int32_t* __restrict__ tok, float* __restrict__ D,
                                   long long N, int w) {
  const long long n = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / 32;
  const int lane = threadIdx.x % 32;
  if (n >= N) return;
  float* dst = D + (long long)tok[n] * w;
  for (int j = lane; j < w; j += 32) {
    const float x = kBf16 ? __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(Xv)[n * w + j])
                          : reinterpret_cast<const float*>(Xv)[n * w + j];
    atomicAdd(dst + j, x);
  }
}

int simt_scatter_add_act_rows(const void* X, int bf16, const int32_t* tok, float* D, long long N, int w, cudaStream_t stream) {
  if (N <= 0) return MAPL_OK;
  KernelScope ks(KID_SCATTER_ROWS, stream);
  const unsigned blocks = (unsigned)((N * 32 + 255) / 256);
  if (bf16) k_scatter_act_rows<true><<<blocks, 256, 0, stream>>>(X, tok, D, N, w);
  else k_scatter_act_rows<false><<<blocks, 256, 0, stream>>>(X, tok, D, N, w);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

__global__ void k_transpose(const float* __restrict__ src, float* __restrict__ dst, int rows, int cols) {
  __shared__ float tile[32][33];
  const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32, tx = threadIdx.x % 32, ty = threadIdx.x / 32;
  for (int i = ty; i < 32; i += 8)
    tile[i][tx] = (r0 + i < rows && c0 + tx < cols) ? src[(long long)(r0 + i) * cols + c0 + tx] : 0.f;
  __syncthreads();
  for (int i = ty; i < 32; i += 8)
    if (c0 + i < cols && r0 + tx < rows) dst[(long long)(c0 + i) * rows + r0 + tx] = tile[tx][i];
}

int simt_transpose(const float* src, float* dst, int rows, int cols, cudaStream_t stream) {
  KernelScope ks(KID_SCATTER_ROWS, stream);
  k_transpose<<<dim3((cols + 31) / 32, (rows + 31) / 32), 256, 0, stream>>>(src, dst, rows, cols);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int simt_half_sqnorm(const float* C, float* out, int rows, int r, cudaStream_t stream) {
  if (rows <= 0) return MAPL_OK;
  const int wpb = 8;
  KernelScope ks(KID_HALF_SQNORM, stream);
  k_half_sqnorm<<<(rows + wpb - 1) / wpb, wpb * 32, 0, stream>>>(C, out, rows, r);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int simt_encode_rvq(const mapl_boundary_desc& d, const void* H, const float* U, const float* C,
                    const float* half_norm, void* Zq_out, int32_t* codes, cudaStream_t stream, const int32_t* tok,
                    const float* Tc) {
  if (d.n_tokens <= 0) return MAPL_OK;
  const int rpad = (d.r + BK - 1) / BK * BK;
  const size_t smem = ((size_t)rpad * LD + 2 * BK * LD) * sizeof(float) + TOK * MAXL * sizeof(int);
  if (smem > 227 * 1024) return MAPL_ERR_UNSUPPORTED;
  const long long blocks = (d.n_tokens + TOK - 1) / TOK;
  KernelScope ks(KID_SIMT_ENCODE_RVQ, stream);
  MAPL_SMEM_OPT_IN(k_simt_encode_rvq<true>, 227 * 1024);
  MAPL_SMEM_OPT_IN(k_simt_encode_rvq<false>, 227 * 1024);
  if (d.act_dtype == MAPL_BF16) {
    k_simt_encode_rvq<true><<<(unsigned)blocks, NT, smem, stream>>>(H, U, C, half_norm, Zq_out, codes, d.n_tokens, d.d, d.r, d.rvq_levels, d.rvq_k, tok, Tc);
  } else {
    k_simt_encode_rvq<false><<<(unsigned)blocks, NT, smem, stream>>>(H, U, C, half_norm, Zq_out, codes, d.n_tokens, d.d, d.r, d.rvq_levels, d.rvq_k, tok, Tc);
  }
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int simt_dequant(const mapl_boundary_desc& d, const int32_t* codes, const float* C, float* Zhat,
                 cudaStream_t stream) {
  const long long total = d.n_tokens * d.r;
  if (total <= 0) return MAPL_OK;
  KernelScope ks(KID_DEQUANT, stream);
  k_dequant<<<(unsigned)((total + 255) / 256), 256, 0, stream>>>(codes, C, Zhat, d.n_tokens, d.r, d.rvq_levels, d.rvq_k);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int simt_scatter_add_rows(const float* gA, const int32_t* tok, float* dA, long long N, int ra,
                          cudaStream_t stream) {
  const long long total = N * ra;
  if (total <= 0) return MAPL_OK;
  KernelScope ks(KID_SCATTER_ROWS, stream);
  if (ra % 4 == 0 && (reinterpret_cast<uintptr_t>(gA) & 15u) == 0 && (reinterpret_cast<uintptr_t>(dA) & 15u) == 0) {
    const long long blocks = (N + 127) / 128;
    k_scatter_add_rows<<<(unsigned)(blocks < 148 * 16 ? blocks : 148 * 16), 128, 0, stream>>>(gA, tok, dA, N, ra);
  } else {
    k_scatter_add_elems<<<(unsigned)((total + 255) / 256), 256, 0, stream>>>(gA, tok, dA, N, ra);
  }
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

}  // namespace mapl
