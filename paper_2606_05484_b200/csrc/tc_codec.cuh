// tc_codec.cuh -- tensor-core (tcgen05 + TMA + TMEM) paths of the codec.  Each tc_* entry returns
// MAPL_ERR_UNSUPPORTED when the boundary is outside its envelope (the caller then runs the fp32
// SIMT kernels), MAPL_OK once everything is enqueued, or an error.
//
// Envelope (v1): bf16 activations, d % 128 == 0, r in {64,128,256}, anchor_rank in {0,64,128}.
// Parameter packs (bf16, rebuilt by every call from the fp32 masters; a few hundred KB):
//   WB [(r+ra), d] = [U^T ; B]    K-major over d     (encode / backward-gz B operand)
//   Wd [d, (r+ra)] = [U | B^T]    K-major over r+ra  (decode / backward-dH B operand)
#pragma once
#include "common.cuh"

namespace mapl {

size_t tc_workspace_bytes(const mapl_boundary_desc& d);
bool tc_shape_ok(const mapl_boundary_desc& d);

struct TcPacks {
  __nv_bfloat16* WB;
  __nv_bfloat16* Wd;
  int kc;   // r + ra
};
TcPacks tc_packs(const mapl_boundary_desc& d, char* tc_ws);
// tokens per CTA (<= 128, multiple of 8) such that the grid covers the 148 SMs in whole, even waves
int tc_tile_m(long long N);
// which: bit0 = WB rows [0,r) (U^T), bit1 = WB rows [r,r+ra) (B), bit2 = Wd cols [0,r) (U), bit3 = Wd cols [r,..) (B^T)
int tc_pack_params(const mapl_boundary_desc& d, const float* U, const float* B, const TcPacks& p, int which,
                   cudaStream_t st);

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
