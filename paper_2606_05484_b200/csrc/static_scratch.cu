// static_scratch.cu -- mapl_encode_rvq_static: the RVQ encode with its scratch in a device array of the library itself,
// for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc) and therefore cannot hand mapl_encode a workspace.
//
// It is mapl_encode on the fp32 SIMT kernels (simt_codec.cu: projection + residual VQ in one kernel, exact fp32
// arithmetic; the path config 0 takes through mapl_encode): the only scratch those need is the table of half squared
// norms 0.5 ||C_l,k||^2, [L*K] fp32, written by k_half_sqnorm and read by k_simt_encode_rvq.  Here that table lives in
// g_half_norm_scratch below -- kStaticScratchRows floats = 64 KB that every GPU which loads the library holds until
// the process exits -- instead of the caller's workspace.  Nothing is allocated, by this file or by what it calls.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address; the address the kernels get
// comes from cudaGetSymbolAddress, asked once per device with that device current (scratch_ptr() below).
//
// Every call on a device shares the one array.  Each call rewrites entries [0, L*K) before it reads them and nothing
// has to start at zero, so the contents a previous call left behind are harmless; but two calls that OVERLAP on the
// GPU (different streams, or graph branches that may run concurrently) race on it.  Serialise them.
#include <mutex>

#include "common.cuh"

namespace mapl {
namespace {

constexpr int kStaticScratchRows = 16384;          // L*K at most: e.g. 4 levels of 4096 codewords, 8 of 2048
static __device__ __align__(256) float g_half_norm_scratch[kStaticScratchRows];

// device address of the array on the CURRENT device; looked up once per device
int scratch_ptr(float** out) {
  static std::mutex mu;
  static float* ptr[kMaxDevices] = {};
  int dev = -1;
  MAPL_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return MAPL_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (ptr[dev] == nullptr) {
    float* p = nullptr;
    MAPL_CUDA_CHECK(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_half_norm_scratch));
    if (p == nullptr) return MAPL_ERR_CUDA;
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return MAPL_OK;
}

}  // namespace
}  // namespace mapl

using namespace mapl;

extern "C" {

size_t mapl_static_scratch_rows(void) { return (size_t)kStaticScratchRows; }

int mapl_encode_rvq_static(const mapl_boundary_desc* desc, const void* H, const float* U, const float* codebooks,
                           void* Zq_out, int32_t* codes_out, void* cuda_stream) {
  if (!desc) return MAPL_ERR_INVALID_ARG;
  const mapl_boundary_desc& d = *desc;
  if (d.n_tokens < 0 || d.d < 8 || d.d % 8 || d.r < 8 || d.r % 8 || d.r > d.d) return MAPL_ERR_INVALID_ARG;
  if (d.act_dtype != MAPL_F32 && d.act_dtype != MAPL_BF16) return MAPL_ERR_INVALID_ARG;
  if (d.rvq_levels < 1 || d.rvq_levels > 8 || d.rvq_k < 1) return MAPL_ERR_INVALID_ARG;       // RVQ on: that is the scratch
  if (d.rvq_group_dim != 0 && d.rvq_group_dim != d.r) return MAPL_ERR_UNSUPPORTED;
  if (d.r > 512 || d.n_tokens > (1ll << 31) - 256) return MAPL_ERR_UNSUPPORTED;
  // the limit of the static array: a clear status instead of writing past it
  if ((long long)d.rvq_levels * d.rvq_k > kStaticScratchRows) return MAPL_ERR_WORKSPACE;
  if (d.n_tokens == 0) return MAPL_OK;
  if (!H || !U || !codebooks || !codes_out) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(H) || !aligned16(U) || !aligned16(codebooks) || !aligned16(codes_out) || (Zq_out && !aligned16(Zq_out)))
    return MAPL_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  float* hn = nullptr;
  MAPL_RETURN_IF(scratch_ptr(&hn));
  MAPL_RETURN_IF(simt_half_sqnorm(codebooks, hn, d.rvq_levels * d.rvq_k, d.r, st));
  return simt_encode_rvq(d, H, U, codebooks, hn, Zq_out, codes_out, st);
}

}  // extern "C"
