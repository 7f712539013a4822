// tc_codec.cuh -- tensor-core (tcgen05 + TMA + TMEM) paths of the codec.  Each function returns
// MAPL_ERR_UNSUPPORTED when the boundary is outside its envelope (the caller then runs the fp32
// SIMT kernels), MAPL_OK once everything is enqueued, or an error.
#pragma once
#include "common.cuh"

namespace mapl {

size_t tc_workspace_bytes(const mapl_boundary_desc& d);

int tc_encode(const mapl_boundary_desc& d, const void* H, const float* U, const float* codebooks,
              void* Zq_out, int32_t* codes_out, char* tc_ws, cudaStream_t st);

int tc_decode(const mapl_boundary_desc& d, const void* Z, const int32_t* codes, const float* U,
              const float* codebooks, const int32_t* tok, const float* A, const float* B, void* Hhat_out,
              char* tc_ws, cudaStream_t st);

// tok == nullptr: anchor ignored.  gA_ws: [N,ra] fp32 scratch.
int tc_backward(const mapl_boundary_desc& d, const void* g, const void* H, const void* Z, const int32_t* codes,
                const float* U, const float* codebooks, const int32_t* tok, const float* A, const float* B,
                void* gz_out, float* dU_out, float* dA_out, float* dB_out, void* dH_out, char* tc_ws,
                float* gA_ws, cudaStream_t st);

}  // namespace mapl
