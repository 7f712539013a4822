// tc_codec.cuh -- tensor-core (tcgen05 + TMA + TMEM) paths of the codec.  Each tc_* entry returns
// MAPL_ERR_UNSUPPORTED when the boundary is outside its envelope (the caller then runs the fp32
// SIMT kernels), MAPL_OK once everything is enqueued, or an error.
//
// Envelope: bf16 activations, d % 256 == 0, r in {64,128,256}, anchor_rank in {0,64,128};
// RVQ on the tensor cores additionally needs K % 128 == 0.
//
// Parameter pack (bf16 operand copies of the fp32 masters, see mapl_pack_params in mapl.h):
//   WB   [(r+ra), d] = [U^T ; B]    K-major over d     (encode / backward-gz B operand)
//   Wd   [d, (r+ra)] = [U | B^T]    K-major over r+ra  (decode / backward-dH B operand)
//   WBlo [r, d]      = bf16(U - bf16(U))^T             (second split term: z to 2^-17 for RVQ)
//   WBlo2 [r, d]     = bf16(U - hi - lo)^T             (third split term, L >= 3 only: z fp32-accurate, so that the deep
//                    levels, whose residual is small against the absolute error of z, stay inside rule S5)
//   Cb   [L*K, r]    fp16 codebooks scaled per level by sc_l = 2^-e (max|c| 2^-e in [0.5,1))
//   hnb  [L*K, 16]   fp16: -(three-term fp16 split of q_k = 0.5 ||C_k||^2 sc_l 2^-g_l), zero padded: the extra K = 16
//                    step of the score MMA that folds the half norms in (tc_encode_rvq.cu)
//   lvl  [8 x 8]     per level: {cmax sc_l, max_k q_k, 2^g_l, sc_l, 2^e, cmax, -, -}, cmax = max_k ||C_l,k||
//   hn   [L*K]       0.5 ||C_k||^2 (fp32), rowamax [L*K]: scratch of the pack kernels
#pragma once
#include "common.cuh"

namespace mapl {

bool tc_shape_ok(const mapl_boundary_desc& d);
bool tc_rvq_ok(const mapl_boundary_desc& d);

struct TcPack {
  __nv_bfloat16* WB = nullptr;
  __nv_bfloat16* Wd = nullptr;
  __nv_bfloat16* WBlo = nullptr;
  __nv_bfloat16* WBlo2 = nullptr;
  __nv_bfloat16* Cb = nullptr;
  __nv_bfloat16* hnb = nullptr;
  float* hn = nullptr;
  float* rowamax = nullptr;
  float* lvl = nullptr;
  int kc = 0;          // r + ra
  size_t bytes = 0;
};
// layout of a pack placed at `base` (base may be nullptr to query `bytes`); bytes == 0 outside the envelope
TcPack tc_pack_layout(const mapl_boundary_desc& d, char* base);
int tc_pack_build(const mapl_boundary_desc& d, const float* U, const float* B, const float* codebooks,
                  const TcPack& p, cudaStream_t st);

// scratch of the tc path besides the pack: bf16 zhat [N,r] (RVQ codes -> dU operand)
size_t tc_scratch_bytes(const mapl_boundary_desc& d);

// global overflow area of the RVQ candidate lists (tc_encode_rvq.cu): kRvqOverflowEntries entries of kRvqOverflowBytes
// per scan thread (256 per CTA); entries are touched only by the rare token whose list in shared memory is full
constexpr int kRvqOverflowEntries = 8;
constexpr int kRvqOverflowBytes = 80;      // m, group id, 2 pad words, 16 raw scores
size_t tc_rvq_overflow_bytes(const mapl_boundary_desc& d);

// tokens per CTA (<= 128, multiple of 8) such that the grid covers the 148 SMs in whole, even waves
int tc_tile_m(long long N);
// the same for kernels launched as clusters of two CTA pairs: only 33 such clusters (132 CTAs) are resident at a time
// (cudaOccupancyMaxActiveClusters on B200: the GPCs do not all hold a multiple of 4 SMs)
int tc_tile_m4(long long N);
// pairs per cluster for decode / backward-gz: 1, or 2 with MAPL_NQ=2 in the environment -- then the two pairs of a
// cluster share every parameter tile by TMA multicast (half the L2 -> SM parameter traffic).  Measured at config 3: no
// gain (decode 59.4 vs 58.9 us, backward 161 vs 163 us) while only 132 CTAs are resident, so it stays opt-in.
int tc_pairs_per_cluster();

// tok / Tc (both or neither): sender-side centring z -= Tc[tok], Tc [V,r] fp32 (mapl_center_table)
// ovf_ws: tc_rvq_overflow_bytes(d) bytes of scratch (RVQ only; nullptr: lists limited to shared memory)
int tc_encode(const mapl_boundary_desc& d, const void* H, const float* codebooks, const TcPack& pk, void* Zq_out,
              int32_t* codes_out, cudaStream_t st, const int32_t* tok = nullptr, const float* Tc = nullptr,
              void* ovf_ws = nullptr);

int tc_decode(const mapl_boundary_desc& d, const void* Z, const int32_t* codes, const float* codebooks,
              const int32_t* tok, const float* A, const TcPack& pk, void* Hhat_out, cudaStream_t st);

// tok == nullptr: anchor ignored.  gA_ws: [N,ra] fp32 scratch; zhat_ws: [N,r] bf16 scratch.
// Zeroes dU/dA/dB itself when accumulate == 0.
int tc_backward(const mapl_boundary_desc& d, const void* g, const void* H, const void* Z, const int32_t* codes,
                const float* codebooks, const int32_t* tok, const float* A, const TcPack& pk, void* gz_out,
                float* dU_out, float* dA_out, float* dB_out, void* dH_out, int accumulate, float* gA_ws,
                __nv_bfloat16* zhat_ws, cudaStream_t st);

}  // namespace mapl
