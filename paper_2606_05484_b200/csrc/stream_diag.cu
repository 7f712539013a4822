// stream_diag.cu -- SURVEY 8f "next" row 4: the device side of the streaming codebook synchronisation
// (Sec. 3.5 "Codebook Synchronization", App. F; reading S15) and the retained-energy
// diagnostic of Fig. 4(b).
//
//   mapl_codebook_delta_pack   rows_out[i, :] = codebooks[idx[i], :]      the subset of codewords a micro-batch carries
//   mapl_codebook_delta_apply  codebooks[idx[i], :] = rows[i, :]          the receiver patches its copy
//        codebooks is viewed as [L*K, r] fp32; idx are flat row numbers.  Which rows travel with which micro-batch is
//        protocol logic of the host (a seeded permutation cut into `interval` parts, reading S15).
//   mapl_energy_retained       out[0] += ||Z||_F^2, out[1] += ||H||_F^2   E = out[0] / out[1] = ||X A||_F^2 / ||X||_F^2
//
// Row copies are pure bandwidth (128-bit accesses); the energy sums are one pass over H and Z with fp32 partial sums
// per thread, fp64 accumulation per block and one atomicAdd(double) per block.
#include "common.cuh"
#include "profile.cuh"

namespace mapl {
namespace {

template <bool kScatter>
__global__ void k_rows_copy(float* __restrict__ table, const int32_t* __restrict__ idx, float* __restrict__ rows, int m, int r) {
  const int vpr = r / 4;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)m * vpr) return;
  const int row = (int)(i / vpr), v = (int)(i % vpr);
  float4* t = reinterpret_cast<float4*>(table + (long long)idx[row] * r) + v;
  float4* p = reinterpret_cast<float4*>(rows + (long long)row * r) + v;
  if (kScatter) *t = *p; else *p = *t;
}

template <bool kBf16>
__global__ void __launch_bounds__(256) k_sumsq(const void* __restrict__ Xv, long long n, double* __restrict__ out) {
  __shared__ double red[8];
  float s = 0.f;
  double acc = 0.0;
  int cnt = 0;
  for (long long i = ((long long)blockIdx.x * 256 + threadIdx.x) * 8; i < n; i += (long long)gridDim.x * 256 * 8) {
    if (kBf16) {
      const uint4 u = *reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(Xv) + i);
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&u);
#pragma unroll
      for (int j = 0; j < 4; ++j) { const float2 f = __bfloat1622float2(h[j]); s = fmaf(f.x, f.x, s); s = fmaf(f.y, f.y, s); }
    } else {
      const float4 a = *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(Xv) + i);
      const float4 b = *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(Xv) + i + 4);
      s = fmaf(a.x, a.x, s); s = fmaf(a.y, a.y, s); s = fmaf(a.z, a.z, s); s = fmaf(a.w, a.w, s);
      s = fmaf(b.x, b.x, s); s = fmaf(b.y, b.y, s); s = fmaf(b.z, b.z, s); s = fmaf(b.w, b.w, s);
    }
    if (++cnt == 64) { acc += (double)s; s = 0.f; cnt = 0; }      // keep the fp32 partial sums short
  }
  acc += (double)s;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (threadIdx.x % 32 == 0) red[threadIdx.x / 32] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < 8; ++k) acc += red[k];
    atomicAdd(out, acc);
  }
}

}  // namespace
}  // namespace mapl

using namespace mapl;

extern "C" {

int mapl_codebook_delta_pack(const float* codebooks, int32_t r, const int32_t* idx, int32_t m, float* rows_out, void* cuda_stream) {
  if (m < 0 || r < 4 || r % 4) return MAPL_ERR_INVALID_ARG;
  if (m == 0) return MAPL_OK;
  if (!codebooks || !idx || !rows_out) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(codebooks) || !aligned16(idx) || !aligned16(rows_out)) return MAPL_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const long long total = (long long)m * (r / 4);
  KernelScope ks(KID_STREAM_DIAG, st);
  k_rows_copy<false><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(const_cast<float*>(codebooks), idx, rows_out, m, r);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int mapl_codebook_delta_apply(float* codebooks_inout, int32_t r, const int32_t* idx, int32_t m, const float* rows, void* cuda_stream) {
  if (m < 0 || r < 4 || r % 4) return MAPL_ERR_INVALID_ARG;
  if (m == 0) return MAPL_OK;
  if (!codebooks_inout || !idx || !rows) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(codebooks_inout) || !aligned16(idx) || !aligned16(rows)) return MAPL_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const long long total = (long long)m * (r / 4);
  KernelScope ks(KID_STREAM_DIAG, st);
  k_rows_copy<true><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(codebooks_inout, idx, const_cast<float*>(rows), m, r);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int mapl_energy_retained(int64_t n_tokens, int32_t d, int32_t r, int32_t act_dtype, const void* H, const void* Z,
                         double* sums_inout, void* cuda_stream) {
  if (n_tokens < 0 || d < 8 || d % 8 || r < 8 || r % 8) return MAPL_ERR_INVALID_ARG;
  if (act_dtype != MAPL_F32 && act_dtype != MAPL_BF16) return MAPL_ERR_INVALID_ARG;
  if (n_tokens == 0) return MAPL_OK;
  if (!H || !Z || !sums_inout) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(H) || !aligned16(Z) || !aligned16(sums_inout)) return MAPL_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  KernelScope ks(KID_STREAM_DIAG, st);
  if (act_dtype == MAPL_BF16) {
    k_sumsq<true><<<148 * 4, 256, 0, st>>>(Z, n_tokens * r, sums_inout);
    k_sumsq<true><<<148 * 4, 256, 0, st>>>(H, n_tokens * d, sums_inout + 1);
  } else {
    k_sumsq<false><<<148 * 4, 256, 0, st>>>(Z, n_tokens * r, sums_inout);
    k_sumsq<false><<<148 * 4, 256, 0, st>>>(H, n_tokens * d, sums_inout + 1);
  }
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

}  // extern "C"
