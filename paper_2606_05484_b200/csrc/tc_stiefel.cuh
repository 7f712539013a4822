// tc_stiefel.cuh -- split-bf16 tensor-core GEMMs of the Stiefel step (tc_stiefel.cu).
#pragma once
#include "common.cuh"

namespace mapl {

// shapes the tensor-core path takes (otherwise the fp32 FFMA kernels of stiefel.cu run)
bool tc_st_ok(int d, int r);
// bytes of the three bf16 planes of `batch` [d,r] matrices
size_t tc_st_plane_bytes(int d, int r, int batch);
// src [batch][rows][cols] fp32 -> planes prow [batch][3][rows][cols] and / or ptr [batch][3][cols][rows]
// mode 0: x;  1: (3 I - x)/2;  2: I + lr (x + x^T)/2;  3: -(x + x^T)/2  (modes 1-3 need rows == cols)
// zero (optional): fp32 buffer of `nzero` elements per batch item (multiple of 4) cleared by the same launch
int tc_st_split(const float* src, int rows, int cols, int batch, int mode, float lr, __nv_bfloat16* prow,
                __nv_bfloat16* ptr, cudaStream_t st, float* zero = nullptr, long long nzero = 0);
// C[b] (+)= A[b] B[b]^T, planes Ap [batch][3][M][K], Bp [batch][3][N][K]; nsplit > 1: split over K with reds
// into a zeroed C; else C = acc + beta E.  M, N multiples of 128, K of 64.
int tc_st_gemm3(const __nv_bfloat16* Ap, const __nv_bfloat16* Bp, int M, int N, int K, int batch, float* C, const float* E,
                float beta, int nsplit, cudaStream_t st);

}  // namespace mapl
