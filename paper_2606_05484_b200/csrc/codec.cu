// codec.cu -- C-ABI entry points mapl_encode / mapl_decode / mapl_codec_backward (include/mapl.h):
// host-side validation, workspace carving and kernel selection.  bf16 boundaries whose shape fits
// the tensor-core envelope run the tcgen05 kernels (tc_*.cu); everything else (fp32 activations,
// ragged shapes) runs the fp32 SIMT kernels.  There is no CPU path.
#include <string.h>

#include "common.cuh"
#include "profile.cuh"
#include "tc_codec.cuh"

namespace mapl {
namespace {

int validate_desc(const mapl_boundary_desc* d) {
  if (!d) return MAPL_ERR_INVALID_ARG;
  if (d->n_tokens < 0) return MAPL_ERR_INVALID_ARG;
  if (d->d < 8 || d->d % 8) return MAPL_ERR_INVALID_ARG;
  if (d->r < 8 || d->r % 8 || d->r > d->d) return MAPL_ERR_INVALID_ARG;
  if (d->act_dtype != MAPL_F32 && d->act_dtype != MAPL_BF16) return MAPL_ERR_INVALID_ARG;
  if (d->rvq_levels < 0 || d->rvq_levels > 8) return MAPL_ERR_INVALID_ARG;
  if (d->rvq_levels > 0 && d->rvq_k < 1) return MAPL_ERR_INVALID_ARG;
  if (d->anchor_rank < 0 || d->anchor_rank % 8) return MAPL_ERR_INVALID_ARG;
  if (d->anchor_rank > 0 && d->vocab < 1) return MAPL_ERR_INVALID_ARG;
  if (d->rvq_levels > 0 && d->rvq_group_dim != 0 && d->rvq_group_dim != d->r) return MAPL_ERR_UNSUPPORTED;
  if (d->rvq_levels > 0 && d->r > 512) return MAPL_ERR_UNSUPPORTED;
  if (d->n_tokens > (1ll << 31) - 256) return MAPL_ERR_UNSUPPORTED;
  return MAPL_OK;
}

// workspace layout (256-byte aligned segments)
struct Ws {
  size_t half_norm = 0;   // [L*K] fp32
  size_t zhat = 0;        // [N*r] fp32 (dequantised codes, SIMT path)
  size_t gA = 0;          // [N*ra] fp32
  size_t pack = 0;        // tensor-core parameter pack, used when desc.param_pack == NULL
  size_t tc = 0;          // tensor-core path scratch (bf16 zhat)
  size_t rvq_ovf = 0;     // overflow area of the RVQ candidate lists (tensor-core encode)
  size_t total = 0;
};

Ws carve(const mapl_boundary_desc& d) {
  Ws w;
  size_t off = 0;
  auto seg = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  w.half_norm = seg((size_t)d.rvq_levels * (size_t)d.rvq_k * 4);
  w.zhat = seg(d.rvq_levels > 0 ? (size_t)d.n_tokens * d.r * 4 : 0);
  w.gA = seg((size_t)d.n_tokens * d.anchor_rank * 4);
  w.pack = seg(tc_pack_layout(d, nullptr).bytes);
  w.tc = seg(tc_scratch_bytes(d));
  w.rvq_ovf = seg(tc_rvq_overflow_bytes(d));
  w.total = off + 256;
  return w;
}

// the parameter pack of this call: the caller's (desc.param_pack) or one built now in the workspace
int resolve_pack(const mapl_boundary_desc& d, const float* U, const float* B, const float* codebooks, char* ws,
                 const Ws& w, cudaStream_t st, TcPack* out) {
  if (d.param_pack) {
    *out = tc_pack_layout(d, const_cast<char*>(reinterpret_cast<const char*>(d.param_pack)));
    return MAPL_OK;
  }
  *out = tc_pack_layout(d, ws + w.pack);
  return tc_pack_build(d, U, B, codebooks, *out, st);
}

bool all16(std::initializer_list<const void*> ps) {
  for (const void* p : ps) if (p && !aligned16(p)) return false;
  return true;
}

}  // namespace
}  // namespace mapl

using namespace mapl;

extern "C" {

const char* mapl_status_string(int status) {
  switch (status) {
    case MAPL_OK: return "MAPL_OK";
    case MAPL_ERR_INVALID_ARG: return "MAPL_ERR_INVALID_ARG";
    case MAPL_ERR_UNSUPPORTED: return "MAPL_ERR_UNSUPPORTED";
    case MAPL_ERR_ALIGNMENT: return "MAPL_ERR_ALIGNMENT";
    case MAPL_ERR_WORKSPACE: return "MAPL_ERR_WORKSPACE";
    case MAPL_ERR_CUDA: return "MAPL_ERR_CUDA";
    default: return "MAPL_ERR_UNKNOWN";
  }
}

const char* mapl_version(void) { return "mapl-b200 0.1 sm_100a"; }

int mapl_last_cuda_error(void) { return g_last_cuda_error; }

size_t mapl_param_pack_bytes(const mapl_boundary_desc* desc) {
  if (validate_desc(desc) != MAPL_OK) return 0;
  return tc_pack_layout(*desc, nullptr).bytes;
}

int mapl_pack_params(const mapl_boundary_desc* desc, const float* U, const float* B, const float* codebooks,
                     void* pack_out, void* cuda_stream) {
  MAPL_RETURN_IF(validate_desc(desc));
  const mapl_boundary_desc& d = *desc;
  const TcPack lay = tc_pack_layout(d, reinterpret_cast<char*>(pack_out));
  if (lay.bytes == 0) return MAPL_OK;                       // fp32 kernels read the masters directly
  if (!U || !pack_out) return MAPL_ERR_INVALID_ARG;
  // B == NULL with anchor_rank > 0 / codebooks == NULL with rvq_levels > 0: that section of an existing pack is
  // left as it is (re-pack after a projector update only)
  if (!all16({U, B, codebooks}) || (reinterpret_cast<uintptr_t>(pack_out) & 255u)) return MAPL_ERR_ALIGNMENT;
  return tc_pack_build(d, U, B, codebooks, lay, reinterpret_cast<cudaStream_t>(cuda_stream));
}

size_t mapl_workspace_bytes(const mapl_boundary_desc* desc) {
  if (validate_desc(desc) != MAPL_OK) return 0;
  return carve(*desc).total;
}

// shared by mapl_encode (tok == Tc == NULL) and mapl_encode_centered
static int encode_impl(const mapl_boundary_desc* desc, const void* H, const float* U, const float* codebooks,
                       const int32_t* tok, const float* Tc, void* Zq_out, int32_t* codes_out, void* workspace,
                       size_t workspace_bytes, void* cuda_stream) {
  MAPL_RETURN_IF(validate_desc(desc));
  const mapl_boundary_desc& d = *desc;
  const int L = d.rvq_levels;
  if (d.n_tokens == 0) return MAPL_OK;           // nothing to do; empty tensors may be NULL
  if (!H || !U) return MAPL_ERR_INVALID_ARG;
  if ((tok == nullptr) != (Tc == nullptr)) return MAPL_ERR_INVALID_ARG;
  if (L == 0 && !Zq_out) return MAPL_ERR_INVALID_ARG;
  if (L > 0 && (!codes_out || !codebooks)) return MAPL_ERR_INVALID_ARG;
  if (!all16({H, U, codebooks, Zq_out, codes_out, workspace, tok, Tc})) return MAPL_ERR_ALIGNMENT;
  const Ws w = carve(d);
  if (!workspace || workspace_bytes < w.total) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = reinterpret_cast<char*>(workspace);

  if (tc_shape_ok(d) && (L == 0 || tc_rvq_ok(d))) {
    TcPack pk;
    MAPL_RETURN_IF(resolve_pack(d, U, nullptr, codebooks, ws, w, st, &pk));
    int s = tc_encode(d, H, codebooks, pk, Zq_out, codes_out, st, tok, Tc, ws + w.rvq_ovf);
    if (s != MAPL_ERR_UNSUPPORTED) return s;
  }

  const int bf = d.act_dtype == MAPL_BF16;
  if (L == 0) {   // Z = H U (- Tc[tok])
    GemmArgs g;
    g.M = (int)d.n_tokens; g.N = d.r; g.K[0] = d.d;
    g.A[0].p = H; g.A[0].bf16 = bf; g.A[0].so = d.d; g.A[0].sk = 1;
    g.B[0].p = U; g.B[0].so = 1; g.B[0].sk = d.r;
    g.C = Zq_out; g.c_bf16 = bf; g.ldc = d.r;
    // centring: T[tok_n] leaves the fp32 accumulator of row n in the GEMM's epilogue, before the one rounding to the
    // activation dtype (mapl.h); a separate pass over a bf16 Z would round U^T h first and lose 2^-9 |U^T h|
    if (Tc) { g.E = Tc; g.lde = d.r; g.beta = -1.f; g.e_gather = tok; }
    return simt_gemm(g, st);
  }
  float* hn = reinterpret_cast<float*>(ws + w.half_norm);
  MAPL_RETURN_IF(simt_half_sqnorm(codebooks, hn, L * d.rvq_k, d.r, st));
  return simt_encode_rvq(d, H, U, codebooks, hn, Zq_out, codes_out, st, tok, Tc);
}

int mapl_encode(const mapl_boundary_desc* desc, const void* H, const float* U, const float* codebooks,
                void* Zq_out, int32_t* codes_out, void* workspace, size_t workspace_bytes,
                void* cuda_stream) {
  return encode_impl(desc, H, U, codebooks, nullptr, nullptr, Zq_out, codes_out, workspace, workspace_bytes, cuda_stream);
}

int mapl_encode_centered(const mapl_boundary_desc* desc, const void* H, const int32_t* tok, const float* center_table,
                         const float* U, const float* codebooks, void* Zq_out, int32_t* codes_out, void* workspace,
                         size_t workspace_bytes, void* cuda_stream) {
  if (!tok || !center_table) return MAPL_ERR_INVALID_ARG;
  return encode_impl(desc, H, U, codebooks, tok, center_table, Zq_out, codes_out, workspace, workspace_bytes, cuda_stream);
}

size_t mapl_center_workspace_bytes(const mapl_boundary_desc* desc) {
  if (validate_desc(desc) != MAPL_OK || desc->anchor_rank <= 0) return 0;
  return align_up((size_t)desc->anchor_rank * desc->r * 4, 256) + 256;
}

int mapl_center_table(const mapl_boundary_desc* desc, const float* A_s, const float* B_s, const float* U,
                      float* table_out, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  MAPL_RETURN_IF(validate_desc(desc));
  const mapl_boundary_desc& d = *desc;
  if (d.anchor_rank <= 0 || d.vocab < 1) return MAPL_ERR_INVALID_ARG;
  if (!A_s || !B_s || !U || !table_out) return MAPL_ERR_INVALID_ARG;
  if (!all16({A_s, B_s, U, table_out, workspace})) return MAPL_ERR_ALIGNMENT;
  if (!workspace || workspace_bytes < mapl_center_workspace_bytes(desc)) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  float* Wc = reinterpret_cast<float*>(workspace);                       // [ra, r] = B_s U
  MAPL_RETURN_IF(st_gemm_nn(B_s, U, Wc, d.anchor_rank, d.r, d.d, st));
  return st_gemm_nn(A_s, Wc, table_out, d.vocab, d.r, d.anchor_rank, st);   // T = A_s (B_s U)   [V, r]
}

namespace {
struct CenterWs { size_t D, Q, Wc, Wct, Ut, total; };
CenterWs center_carve(const mapl_boundary_desc& d) {
  CenterWs w;
  size_t off = 0;
  auto seg = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  w.D = seg((size_t)d.vocab * d.r * 4);
  w.Q = seg((size_t)d.anchor_rank * d.r * 4);
  w.Wc = seg((size_t)d.anchor_rank * d.r * 4);
  w.Wct = seg((size_t)d.anchor_rank * d.r * 4);
  w.Ut = seg((size_t)d.d * d.r * 4);
  w.total = off + 256;
  return w;
}
}  // namespace

size_t mapl_center_backward_workspace_bytes(const mapl_boundary_desc* desc) {
  if (validate_desc(desc) != MAPL_OK || desc->anchor_rank <= 0 || desc->vocab < 1) return 0;
  return center_carve(*desc).total;
}

int mapl_center_backward(const mapl_boundary_desc* desc, const void* gz, const int32_t* tok, const float* A_s,
                         const float* B_s, const float* U, float* dA_s_out, float* dB_s_out, float* dU_inout,
                         int accumulate, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  MAPL_RETURN_IF(validate_desc(desc));
  const mapl_boundary_desc& d = *desc;
  if (d.anchor_rank <= 0 || d.vocab < 1) return MAPL_ERR_INVALID_ARG;
  if (!A_s || !B_s || !U || !dA_s_out || !dU_inout) return MAPL_ERR_INVALID_ARG;
  if (d.n_tokens > 0 && (!gz || !tok)) return MAPL_ERR_INVALID_ARG;
  if (!all16({gz, tok, A_s, B_s, U, dA_s_out, dB_s_out, dU_inout, workspace})) return MAPL_ERR_ALIGNMENT;
  const CenterWs w = center_carve(d);
  if (!workspace || workspace_bytes < w.total) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = reinterpret_cast<char*>(workspace);
  float* D = reinterpret_cast<float*>(ws + w.D);       // [V,r]  D[v] = sum_{n: tok_n = v} gz_n
  float* Q = reinterpret_cast<float*>(ws + w.Q);       // [ra,r] A_s^T D = sum_n A_s[tok_n] (outer) gz_n
  float* Wc = reinterpret_cast<float*>(ws + w.Wc);     // [ra,r] B_s U
  float* Wct = reinterpret_cast<float*>(ws + w.Wct);   // [r,ra]
  float* Ut = reinterpret_cast<float*>(ws + w.Ut);     // [r,d]
  const int V = d.vocab, ra = d.anchor_rank, r = d.r, dd = d.d;
  { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(D, 0, (size_t)V * r * 4, st)); }
  { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(Q, 0, (size_t)ra * r * 4, st)); }
  MAPL_RETURN_IF(simt_scatter_add_act_rows(gz, d.act_dtype == MAPL_BF16, tok, D, d.n_tokens, r, st));
  MAPL_RETURN_IF(st_gemm_nn(B_s, U, Wc, ra, r, dd, st));
  MAPL_RETURN_IF(simt_transpose(Wc, Wct, ra, r, st));
  MAPL_RETURN_IF(st_gemm_tn(A_s, D, Q, ra, r, V, st));                                        // Q = A_s^T D
  MAPL_RETURN_IF(st_gemm_nn(D, Wct, dA_s_out, V, ra, r, st, -1.f, accumulate ? dA_s_out : nullptr, 1.f));   // dA_s = -D Wc^T
  MAPL_RETURN_IF(st_gemm_tn(B_s, Q, dU_inout, dd, r, ra, st, -1.f));                         // dU += -B_s^T Q
  if (dB_s_out) {
    MAPL_RETURN_IF(simt_transpose(U, Ut, dd, r, st));
    MAPL_RETURN_IF(st_gemm_nn(Q, Ut, dB_s_out, ra, dd, r, st, -1.f, accumulate ? dB_s_out : nullptr, 1.f));   // dB_s = -Q U^T
  }
  return MAPL_OK;
}

int mapl_decode(const mapl_boundary_desc* desc, const void* Z, const int32_t* codes, const float* U,
                const float* codebooks, const int32_t* tok, const float* A, const float* B,
                void* Hhat_out, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  MAPL_RETURN_IF(validate_desc(desc));
  const mapl_boundary_desc& d = *desc;
  if (d.n_tokens == 0) return MAPL_OK;
  if (!U || !Hhat_out) return MAPL_ERR_INVALID_ARG;
  if ((Z == nullptr) == (codes == nullptr)) return MAPL_ERR_INVALID_ARG;
  if (codes && (d.rvq_levels == 0 || !codebooks)) return MAPL_ERR_INVALID_ARG;
  const bool anchor = d.anchor_rank > 0;
  if (anchor && (!tok || !A || !B)) return MAPL_ERR_INVALID_ARG;
  if (!all16({Z, codes, U, codebooks, tok, A, B, Hhat_out, workspace})) return MAPL_ERR_ALIGNMENT;
  const Ws w = carve(d);
  if (!workspace || workspace_bytes < w.total) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = reinterpret_cast<char*>(workspace);

  if (tc_shape_ok(d)) {
    TcPack pk;
    MAPL_RETURN_IF(resolve_pack(d, U, B, codebooks, ws, w, st, &pk));
    int s = tc_decode(d, Z, codes, codebooks, tok, A, pk, Hhat_out, st);
    if (s != MAPL_ERR_UNSUPPORTED) return s;
  }

  const int bf = d.act_dtype == MAPL_BF16;
  GemmArgs g;
  g.M = (int)d.n_tokens; g.N = d.d;
  if (codes) {
    float* zh = reinterpret_cast<float*>(ws + w.zhat);
    MAPL_RETURN_IF(simt_dequant(d, codes, codebooks, zh, st));
    g.A[0].p = zh; g.A[0].bf16 = 0;
  } else {
    g.A[0].p = Z; g.A[0].bf16 = bf;
  }
  g.A[0].so = d.r; g.A[0].sk = 1; g.K[0] = d.r;
  g.B[0].p = U; g.B[0].so = d.r; g.B[0].sk = 1;           // B(k,n) = U[n,k]
  if (anchor) {
    g.npairs = 2; g.K[1] = d.anchor_rank;
    g.A[1].p = A; g.A[1].so = d.anchor_rank; g.A[1].sk = 1; g.A[1].gather = tok; g.A[1].gmode = 1;
    g.B[1].p = B; g.B[1].so = 1; g.B[1].sk = d.d;          // B(k,n) = B[k,n]
  }
  g.C = Hhat_out; g.c_bf16 = bf; g.ldc = d.d;
  return simt_gemm(g, st);
}

int mapl_codec_backward(const mapl_boundary_desc* desc, const void* g_Hhat, const void* H, const void* Z,
                        const int32_t* codes, const float* U, const float* codebooks, const int32_t* tok,
                        const float* A, const float* B, void* gz_out, float* dU_out, float* dA_out,
                        float* dB_out, void* dH_out, int accumulate, void* workspace,
                        size_t workspace_bytes, void* cuda_stream) {
  MAPL_RETURN_IF(validate_desc(desc));
  const mapl_boundary_desc& d = *desc;
  if (d.n_tokens == 0) {                          // only the overwrite semantics remain
    cudaStream_t st0 = reinterpret_cast<cudaStream_t>(cuda_stream);
    if (!accumulate) {
      if (dU_out) MAPL_CUDA_CHECK(cudaMemsetAsync(dU_out, 0, (size_t)d.d * d.r * 4, st0));
      if (dA_out) MAPL_CUDA_CHECK(cudaMemsetAsync(dA_out, 0, (size_t)d.vocab * d.anchor_rank * 4, st0));
      if (dB_out) MAPL_CUDA_CHECK(cudaMemsetAsync(dB_out, 0, (size_t)d.anchor_rank * d.d * 4, st0));
    }
    return MAPL_OK;
  }
  if (!g_Hhat || !U || !gz_out || !dU_out) return MAPL_ERR_INVALID_ARG;
  if ((Z == nullptr) == (codes == nullptr)) return MAPL_ERR_INVALID_ARG;
  if (codes && (d.rvq_levels == 0 || !codebooks)) return MAPL_ERR_INVALID_ARG;
  if (!H && dH_out) return MAPL_ERR_INVALID_ARG;
  bool anchor = d.anchor_rank > 0;
  if (anchor && !tok && !A && !B) anchor = false;           // anchor ignored on request
  if (anchor && (!tok || !A || !B || !dA_out)) return MAPL_ERR_INVALID_ARG;
  if (!anchor && (dA_out || dB_out)) return MAPL_ERR_INVALID_ARG;
  if (!all16({g_Hhat, H, Z, codes, U, codebooks, tok, A, B, gz_out, dU_out, dA_out, dB_out, dH_out, workspace}))
    return MAPL_ERR_ALIGNMENT;
  const Ws w = carve(d);
  if (!workspace || workspace_bytes < w.total) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = reinterpret_cast<char*>(workspace);
  const long long N = d.n_tokens;
  const int ra = anchor ? d.anchor_rank : 0;

  if (tc_shape_ok(d)) {
    TcPack pk;
    MAPL_RETURN_IF(resolve_pack(d, U, anchor ? B : nullptr, codebooks, ws, w, st, &pk));
    int s = tc_backward(d, g_Hhat, H, Z, codes, codebooks, anchor ? tok : nullptr, A, pk, gz_out, dU_out, dA_out,
                        dB_out, dH_out, accumulate, reinterpret_cast<float*>(ws + w.gA),
                        reinterpret_cast<__nv_bfloat16*>(ws + w.tc), st);
    if (s != MAPL_ERR_UNSUPPORTED) return s;
  }
  if (!accumulate) {
    { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(dU_out, 0, (size_t)d.d * d.r * 4, st)); }
    if (anchor) { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(dA_out, 0, (size_t)d.vocab * ra * 4, st)); }
    if (anchor && dB_out) { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(dB_out, 0, (size_t)ra * d.d * 4, st)); }
  }

  const int bf = d.act_dtype == MAPL_BF16;
  // zhat operand
  MatRef zh;
  if (codes) {
    float* z = reinterpret_cast<float*>(ws + w.zhat);
    MAPL_RETURN_IF(simt_dequant(d, codes, codebooks, z, st));
    zh.p = z; zh.bf16 = 0;
  } else {
    zh.p = Z; zh.bf16 = bf;
  }
  {  // gz = g U
    GemmArgs g;
    g.M = (int)N; g.N = d.r; g.K[0] = d.d;
    g.A[0].p = g_Hhat; g.A[0].bf16 = bf; g.A[0].so = d.d; g.A[0].sk = 1;
    g.B[0].p = U; g.B[0].so = 1; g.B[0].sk = d.r;
    g.C = gz_out; g.c_bf16 = bf; g.ldc = d.r;
    MAPL_RETURN_IF(simt_gemm(g, st));
  }
  // split the token contraction so that tiles x splits covers about two waves of the 148 SMs (>= 64 tokens each)
  auto splits_for = [&](int m, int n) {
    const long long tiles = (long long)((m + 63) / 64) * ((n + 63) / 64);
    long long sp = (2 * 148 + tiles - 1) / tiles;
    const long long max_sp = (N + 63) / 64;
    if (sp > max_sp) sp = max_sp;
    return (int)(sp < 1 ? 1 : sp);
  };
  {  // dU += g^T zhat (+ H^T gz)
    GemmArgs g;
    g.M = d.d; g.N = d.r; g.K[0] = (int)N;
    g.A[0].p = g_Hhat; g.A[0].bf16 = bf; g.A[0].so = 1; g.A[0].sk = d.d;
    g.B[0] = zh; g.B[0].so = 1; g.B[0].sk = d.r;
    if (H) {
      g.npairs = 2; g.K[1] = (int)N;
      g.A[1].p = H; g.A[1].bf16 = bf; g.A[1].so = 1; g.A[1].sk = d.d;
      g.B[1].p = gz_out; g.B[1].bf16 = bf; g.B[1].so = 1; g.B[1].sk = d.r;
    }
    g.C = dU_out; g.ldc = d.r; g.atomic = 1; g.splits = splits_for(d.d, d.r);
    MAPL_RETURN_IF(simt_gemm(g, st));
  }
  if (dH_out) {  // dH = gz U^T
    GemmArgs g;
    g.M = (int)N; g.N = d.d; g.K[0] = d.r;
    g.A[0].p = gz_out; g.A[0].bf16 = bf; g.A[0].so = d.r; g.A[0].sk = 1;
    g.B[0].p = U; g.B[0].so = d.r; g.B[0].sk = 1;
    g.C = dH_out; g.c_bf16 = bf; g.ldc = d.d;
    MAPL_RETURN_IF(simt_gemm(g, st));
  }
  if (anchor) {
    float* gA = reinterpret_cast<float*>(ws + w.gA);
    {  // gA = g B^T
      GemmArgs g;
      g.M = (int)N; g.N = ra; g.K[0] = d.d;
      g.A[0].p = g_Hhat; g.A[0].bf16 = bf; g.A[0].so = d.d; g.A[0].sk = 1;
      g.B[0].p = B; g.B[0].so = d.d; g.B[0].sk = 1;
      g.C = gA; g.ldc = ra;
      MAPL_RETURN_IF(simt_gemm(g, st));
    }
    MAPL_RETURN_IF(simt_scatter_add_rows(gA, tok, dA_out, N, ra, st));
    if (dB_out) {  // dB += A[tok]^T g
      GemmArgs g;
      g.M = ra; g.N = d.d; g.K[0] = (int)N;
      g.A[0].p = A; g.A[0].so = 1; g.A[0].sk = ra; g.A[0].gather = tok; g.A[0].gmode = 2;
      g.B[0].p = g_Hhat; g.B[0].bf16 = bf; g.B[0].so = 1; g.B[0].sk = d.d;
      g.C = dB_out; g.ldc = d.d; g.atomic = 1; g.splits = splits_for(ra, d.d);
      MAPL_RETURN_IF(simt_gemm(g, st));
    }
  }
  return MAPL_OK;
}

}  // extern "C"
