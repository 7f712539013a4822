// mcvq.cu -- grouped multi-codebook VQ of a wire payload (Sec. 3.5; reading S3;
// SURVEY 8f "next" row 3): the r channels of every token are cut into r/G groups of G = 2 consecutive channels, each
// group is residual-vector-quantised on its own over L rounds with the 2-dimensional codewords C[l, k, 2g:2g+2], and
// the index is one byte (K <= 256): (r/G) L bytes per token -- 256 B at the paper's r = 256, G = 2, K = 256, R = 2.
// It quantises a stored payload tensor ([N,r] in the activation dtype): the forward payload Z written by mapl_encode,
// or the backward payload gz of mapl_codec_backward ("compressing both forward activations and backward gradients").
//
// N (r/G) L K two-dimensional distance evaluations: CUDA-core work (no contraction worth a tensor core: K = 2 would be
// padded 8x, and the arg-min scan stays on the ALUs anyway), bound by FP32 issue rate.
//   k_mcvq_quantize   CTA = 64 tokens x 8 group lanes (256 threads, two tokens per thread).  Per step the 8 groups'
//                     codeword slices of all rounds (L K float2 each) are staged in shared memory; a warp holds tokens
//                     of ONE group, so every codeword read is a broadcast, shared by two distance evaluations.  Distances in the direct form (x - c)^2, fp32; lowest index
//                     wins ties (S4).
//   k_mcvq_dequantize thread = (token, group): sum of the chosen 2-d codewords, rounded once to the activation dtype.
#include <float.h>

#include "common.cuh"
#include "profile.cuh"

namespace mapl {
namespace {

constexpr int kTok = 64, kLanes = 8, kThreads = 256, kMaxLK = 4 * 256;    // L K <= 1024 codewords per group in shared memory

template <bool kBf16>
__device__ __forceinline__ void load2(const void* Xv, long long off, float* x0, float* x1) {
  if (kBf16) {
    const __nv_bfloat162 v = *reinterpret_cast<const __nv_bfloat162*>(reinterpret_cast<const __nv_bfloat16*>(Xv) + off);
    *x0 = __bfloat162float(v.x); *x1 = __bfloat162float(v.y);
  } else {
    const float2 v = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(Xv) + off);
    *x0 = v.x; *x1 = v.y;
  }
}
template <bool kBf16>
__device__ __forceinline__ void store2(void* Xqv, long long off, float q0, float q1) {
  if (kBf16) *reinterpret_cast<__nv_bfloat162*>(reinterpret_cast<__nv_bfloat16*>(Xqv) + off) = __floats2bfloat162_rn(q0, q1);
  else *reinterpret_cast<float2*>(reinterpret_cast<float*>(Xqv) + off) = make_float2(q0, q1);
}

// CTA = 64 tokens x 8 group lanes, 256 threads: thread (token pair, lane) scans for TWO tokens (n, n + 32) at once, so
// every broadcast codeword read serves two distance evaluations and the two arg-min chains interleave.
template <bool kBf16>
__global__ void __launch_bounds__(kThreads) k_mcvq_quantize(const void* __restrict__ Xv, const float* __restrict__ C,
                                                           uint8_t* __restrict__ codes, void* __restrict__ Xqv, long long N,
                                                           int r, int L, int K) {
  extern __shared__ float2 sC[];                 // [kLanes][L*K]
  const int t = threadIdx.x, tok_l = t % 32, gl = t / 32, ng = r / 2;
  const long long na = (long long)blockIdx.x * kTok + tok_l, nb = na + 32;
  const bool la = na < N, lb = nb < N;
  for (int g0 = 0; g0 < ng; g0 += kLanes) {
    // stage the slices of groups g0 .. g0+7: C[l, k, 2g : 2g+2]
    for (int i = t; i < kLanes * L * K; i += kThreads) {
      const int lane_g = i / (L * K), lk = i % (L * K), g = g0 + lane_g;
      sC[i] = g < ng ? *reinterpret_cast<const float2*>(C + (long long)lk * r + 2 * g) : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const int g = g0 + gl;
    if (g < ng && la) {
      float xa0, xa1, xb0 = 0.f, xb1 = 0.f;
      load2<kBf16>(Xv, na * r + 2 * g, &xa0, &xa1);
      if (lb) load2<kBf16>(Xv, nb * r + 2 * g, &xb0, &xb1);
      float qa0 = 0.f, qa1 = 0.f, qb0 = 0.f, qb1 = 0.f;
      const float2* cg = sC + (size_t)gl * L * K;
      for (int l = 0; l < L; ++l) {
        float besta = FLT_MAX, bestb = FLT_MAX;
        int ka = 0, kb = 0;
        const float2* cl = cg + l * K;
#pragma unroll 8
        for (int k = 0; k < K; ++k) {
          const float2 c = cl[k];
          const float da0 = xa0 - c.x, da1 = xa1 - c.y, db0 = xb0 - c.x, db1 = xb1 - c.y;
          const float dista = fmaf(da1, da1, da0 * da0), distb = fmaf(db1, db1, db0 * db0);
          if (dista < besta) { besta = dista; ka = k; }       // strict: lowest index on ties
          if (distb < bestb) { bestb = distb; kb = k; }
        }
        const float2 ca = cl[ka], cb = cl[kb];
        xa0 -= ca.x; xa1 -= ca.y; qa0 += ca.x; qa1 += ca.y;
        xb0 -= cb.x; xb1 -= cb.y; qb0 += cb.x; qb1 += cb.y;
        codes[(na * L + l) * ng + g] = (uint8_t)ka;
        if (lb) codes[(nb * L + l) * ng + g] = (uint8_t)kb;
      }
      if (Xqv != nullptr) {
        store2<kBf16>(Xqv, na * r + 2 * g, qa0, qa1);
        if (lb) store2<kBf16>(Xqv, nb * r + 2 * g, qb0, qb1);
      }
    }
    __syncthreads();
  }
}

template <bool kBf16>
__global__ void k_mcvq_dequantize(const uint8_t* __restrict__ codes, const float* __restrict__ C, void* __restrict__ Xqv,
                                  long long N, int r, int L, int K) {
  const int ng = r / 2;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * ng) return;
  const long long n = idx / ng;
  const int g = (int)(idx % ng);
  float q0 = 0.f, q1 = 0.f;
  for (int l = 0; l < L; ++l) {
    const int k = codes[(n * L + l) * ng + g];
    const float2 c = *reinterpret_cast<const float2*>(C + ((long long)l * K + k) * r + 2 * g);
    q0 += c.x; q1 += c.y;
  }
  if (kBf16) *reinterpret_cast<__nv_bfloat162*>(reinterpret_cast<__nv_bfloat16*>(Xqv) + n * r + 2 * g) = __floats2bfloat162_rn(q0, q1);
  else *reinterpret_cast<float2*>(reinterpret_cast<float*>(Xqv) + n * r + 2 * g) = make_float2(q0, q1);
}

int check(int64_t N, int r, int L, int K, int act_dtype) {
  if (N < 0 || r < 2 || r % 8 || L < 1 || L > 4 || K < 1 || K > 256) return MAPL_ERR_INVALID_ARG;
  if (L * K > kMaxLK) return MAPL_ERR_UNSUPPORTED;
  if (act_dtype != MAPL_F32 && act_dtype != MAPL_BF16) return MAPL_ERR_INVALID_ARG;
  return MAPL_OK;
}

}  // namespace
}  // namespace mapl

using namespace mapl;

extern "C" {

int mapl_mcvq_quantize(int64_t n_tokens, int32_t r, int32_t act_dtype, int32_t levels, int32_t k, const void* X,
                       const float* codebooks, uint8_t* codes_out, void* Xq_out, void* cuda_stream) {
  MAPL_RETURN_IF(check(n_tokens, r, levels, k, act_dtype));
  if (n_tokens == 0) return MAPL_OK;
  if (!X || !codebooks || !codes_out) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(codebooks) || !aligned16(codes_out) || (Xq_out && !aligned16(Xq_out))) return MAPL_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const size_t smem = (size_t)kLanes * levels * k * sizeof(float2);
  MAPL_SMEM_OPT_IN(k_mcvq_quantize<true>, kLanes * kMaxLK * 8);
  MAPL_SMEM_OPT_IN(k_mcvq_quantize<false>, kLanes * kMaxLK * 8);
  const unsigned blocks = (unsigned)((n_tokens + kTok - 1) / kTok);
  KernelScope ks(KID_MCVQ, st);
  if (act_dtype == MAPL_BF16) k_mcvq_quantize<true><<<blocks, kThreads, smem, st>>>(X, codebooks, codes_out, Xq_out, n_tokens, r, levels, k);
  else k_mcvq_quantize<false><<<blocks, kThreads, smem, st>>>(X, codebooks, codes_out, Xq_out, n_tokens, r, levels, k);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int mapl_mcvq_dequantize(int64_t n_tokens, int32_t r, int32_t act_dtype, int32_t levels, int32_t k, const uint8_t* codes,
                         const float* codebooks, void* Xq_out, void* cuda_stream) {
  MAPL_RETURN_IF(check(n_tokens, r, levels, k, act_dtype));
  if (n_tokens == 0) return MAPL_OK;
  if (!codes || !codebooks || !Xq_out) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(codes) || !aligned16(codebooks) || !aligned16(Xq_out)) return MAPL_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const long long total = n_tokens * (r / 2);
  KernelScope ks(KID_MCVQ, st);
  if (act_dtype == MAPL_BF16) k_mcvq_dequantize<true><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(codes, codebooks, Xq_out, n_tokens, r, levels, k);
  else k_mcvq_dequantize<false><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(codes, codebooks, Xq_out, n_tokens, r, levels, k);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

}  // extern "C"
