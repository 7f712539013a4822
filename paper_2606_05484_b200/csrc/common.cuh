// common.cuh -- shared host/device helpers of libmapl (CUDA path only; the oracle shares nothing).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "mapl.h"

namespace mapl {

extern thread_local int g_last_cuda_error;

#define MAPL_CUDA_CHECK(expr)                      \
  do {                                             \
    cudaError_t e_ = (expr);                       \
    if (e_ != cudaSuccess) {                       \
      ::mapl::g_last_cuda_error = (int)e_;         \
      return MAPL_ERR_CUDA;                        \
    }                                              \
  } while (0)

#define MAPL_RETURN_IF(expr)        \
  do {                              \
    int s_ = (expr);                \
    if (s_ != MAPL_OK) return s_;   \
  } while (0)

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a per-DEVICE property of a kernel: set it once per device the
// process drives, under a lock (two host threads may make their first call together).  Usage:
//   MAPL_SMEM_OPT_IN(k_tc_decode, 227 * 1024);
#define MAPL_SMEM_OPT_IN(kernel, bytes)                                                                    \
  do {                                                                                                     \
    static std::mutex mu_;                                                                                 \
    static bool done_[::mapl::kMaxDevices] = {};                                                           \
    int dev_ = 0;                                                                                          \
    MAPL_CUDA_CHECK(cudaGetDevice(&dev_));                                                                 \
    std::lock_guard<std::mutex> lk_(mu_);                                                                  \
    if (dev_ < 0 || dev_ >= ::mapl::kMaxDevices || !done_[dev_]) {                                         \
      MAPL_CUDA_CHECK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (bytes))); \
      if (dev_ >= 0 && dev_ < ::mapl::kMaxDevices) done_[dev_] = true;                                     \
    }                                                                                                      \
  } while (0)
constexpr int kMaxDevices = 64;

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t act_bytes(int act_dtype) { return act_dtype == MAPL_BF16 ? 2 : 4; }

// ---------------------------------------------------------------- generic SIMT GEMM (fp32 FFMA)
// C[M,N] = alpha * sum_p A_p(m,k) B_p(k,n)  (+ beta * E[m,n]),  element (i,k) of an operand lives at
// p[i*so + k*sk] (after the optional gather of i or k through an int32 index array).
struct MatRef {
  const void* p = nullptr;
  int bf16 = 0;             // 0: fp32 elements, 1: bf16 elements
  long long so = 0;         // stride of the non-contracted index (m for A, n for B)
  long long sk = 0;         // stride of the contracted index k
  long long sb = 0;         // batch stride (elements)
  const int32_t* gather = nullptr;
  int gmode = 0;            // 0 none; 1: outer index i -> gather[i]; 2: k -> gather[k]
};

struct GemmArgs {
  int M = 0, N = 0;
  int npairs = 1;
  MatRef A[2], B[2];
  int K[2] = {0, 0};
  void* C = nullptr;
  int c_bf16 = 0;
  long long ldc = 0, sbc = 0;
  int splits = 1;           // split-K factor (needs atomic when > 1)
  int atomic = 0;           // atomicAdd into fp32 C (C pre-zeroed or accumulating)
  float alpha = 1.f;
  const float* E = nullptr; // optional epilogue matrix (fp32, same indexing as C), only when !atomic
  long long lde = 0, sbe = 0;
  float beta = 0.f;
  const int32_t* e_gather = nullptr;  // optional: row m of E is E[e_gather[m]] (the centring rows T[tok_n] of Eq. 1)
  int batch = 1;
};

int simt_gemm(const GemmArgs& g, cudaStream_t stream);

// C[M,N] = A[M,K] B[K,N], all dense row-major fp32 (the 64x64-tile FFMA kernel of stiefel.cu); N, K % 4 == 0
int st_gemm_nn(const float* A, const float* B, float* C, int M, int N, int K, cudaStream_t stream, float alpha = 1.f,
               const float* E = nullptr, float beta = 0.f);       // C = alpha A B + beta E (E may be C)
// C[M,N] += alpha X[K,M]^T Y[K,N] (split over K, red.global.add: C must hold the value to add to); M, N % 4 == 0
int st_gemm_tn(const float* X, const float* Y, float* C, int M, int N, int K, cudaStream_t stream, float alpha = 1.f);
// D[tok_n, :] += X[n, :] (X in the activation dtype, D fp32 [V,w]);  dst[c, r] = src[r, c] (fp32)
int simt_scatter_add_act_rows(const void* X, int bf16, const int32_t* tok, float* D, long long N, int w, cudaStream_t stream);
int simt_transpose(const float* src, float* dst, int rows, int cols, cudaStream_t stream);

// ---------------------------------------------------------------- SIMT codec pieces (simt_codec.cu)
int simt_half_sqnorm(const float* C, float* out, int rows, int r, cudaStream_t stream);
int simt_encode_rvq(const mapl_boundary_desc& d, const void* H, const float* U, const float* C,
                    const float* half_norm, void* Zq_out, int32_t* codes, cudaStream_t stream,
                    const int32_t* tok = nullptr, const float* Tc = nullptr);     // Tc: centring table (Eq. 1)
int simt_dequant(const mapl_boundary_desc& d, const int32_t* codes, const float* C, float* Zhat,
                 cudaStream_t stream);
int simt_scatter_add_rows(const float* gA, const int32_t* tok, float* dA, long long N, int ra,
                          cudaStream_t stream);

// ---------------------------------------------------------------- tensor-core (tcgen05) paths (tc_*.cu)
// Each returns MAPL_ERR_UNSUPPORTED when the shape is outside its envelope; the caller then
// uses the SIMT kernels above.
bool tc_available();

// ---------------------------------------------------------------- device helpers
#ifdef __CUDACC__
__device__ __forceinline__ float ld_as_f32(const void* p, long long idx, int is_bf16) {
  if (is_bf16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[idx]);
  return reinterpret_cast<const float*>(p)[idx];
}
__device__ __forceinline__ void st_from_f32(void* p, long long idx, int is_bf16, float v) {
  if (is_bf16) reinterpret_cast<__nv_bfloat16*>(p)[idx] = __float2bfloat16_rn(v);
  else reinterpret_cast<float*>(p)[idx] = v;
}
#endif

}  // namespace mapl
