// profile.cuh -- launch accounting of libmapl: every kernel launch site is wrapped in a KernelScope,
// which counts the launch and, when timing is switched on (mapl_profile_enable), brackets it with a
// CUDA-event pair on the launching stream.  Diagnostics only; host-side, not thread-safe.
#pragma once
#include <cuda_runtime.h>

namespace mapl {

enum KernelId {
  KID_SIMT_GEMM = 0,
  KID_HALF_SQNORM,
  KID_SIMT_ENCODE_RVQ,
  KID_DEQUANT,
  KID_SCATTER_ROWS,
  KID_ST_STEP_MATRIX,
  KID_ST_NS_POLY,
  KID_ST_FRO_NORM,
  KID_ST_CHOL,
  KID_ST_TRI_INV,
  KID_MEMSET,
  KID_TC_PACK,
  KID_TC_ENCODE,
  KID_TC_DECODE,
  KID_TC_BWD_GZ,
  KID_TC_BWD_DU,
  KID_TC_ENCODE_RVQ,
  KID_TC_SCATTER,
  KID_ST_GEMM,
  KID_ST_SPLIT,
  KID_ST_GEMM3,
  KID_MCVQ,
  KID_STREAM_DIAG,
  KID_COUNT
};

void prof_begin(int kid, cudaStream_t st);
void prof_end(int kid, cudaStream_t st);

struct KernelScope {
  int kid; cudaStream_t st;
  KernelScope(int k, cudaStream_t s) : kid(k), st(s) { prof_begin(k, s); }
  ~KernelScope() { prof_end(kid, st); }
};

}  // namespace mapl
