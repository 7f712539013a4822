/* mapl.h -- C ABI of the B200-native MAPL boundary codec (libmapl.so).
 *
 * MAPL = Manifold Aware Projection Learning, arxiv/paper_2606_05484.  Citations "P:NN" are line NN
 * of the paper text; "S#" are the readings listed in DESIGN.md.
 *
 * The library implements, as hand-written sm_100a CUDA kernels, the per-token pipeline-stage
 * boundary codec and the step that keeps its projector on the Stiefel manifold:
 *
 *   mapl_encode          z = U^T h                          (Eq. 1, Alg. 1 l.1; centring = S6)
 *                        + residual VQ of z                 (Sec. 3.5)
 *   mapl_decode          hhat = U zhat + A[tok] B           (Eq. 2, Alg. 1 l.3, Eq. 3)
 *   mapl_codec_backward  gz = U^T g, dU, dA, dB, dH         (Alg. 1 l.4; STE = S7)
 *   mapl_stiefel_step    xi = G - U sym(U^T G); U <- Retr(U - lr xi)   (Eq. 4, Eq. 7)
 *
 * Notation (paper -> here): X^{b_p} -> H [N,d]; A_p -> U [d,r]; Z^{b_p} -> Z [N,r];
 * E^small -> A [V,ra]; P_p -> B [ra,d]; t_ids -> tok [N]; C_p -> codebooks [L,K,r].
 *
 * GENERAL CONVENTIONS
 *  - Layout: every tensor is dense row-major (row stride == row length).  Row-vector form:
 *    Z = H U, Hhat = Zhat U^T + A[tok] B.
 *  - Memory: unless a parameter says HOST, every pointer is a DEVICE pointer owned by the caller
 *    (allocate with torch / cudaMalloc).  The library never allocates, frees or keeps a pointer
 *    after the call returns.  Descriptors are host structs read during the call only.
 *  - Alignment: every non-NULL device pointer must be 16-byte aligned.
 *  - Dtypes: U, codebooks, A, B, dU, dA, dB and everything in mapl_stiefel_step are fp32.
 *    Activations (H, Hhat, g, dH, Z, gz) have desc.act_dtype (fp32 or bf16).  codes, tok: int32.
 *  - Execution: all work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL =
 *    the legacy default stream).  No host synchronisation, no host read of device data.
 *  - Errors: every entry point returns a mapl_status (0 = OK, negative = error).  On an argument
 *    error nothing is enqueued.  No exception crosses the ABI.  CUDA launch failures map to
 *    MAPL_ERR_CUDA (mapl_last_cuda_error() gives the cudaError_t).
 *  - Preconditions the host cannot check without a sync (the caller's responsibility):
 *    0 <= tok[n] < vocab, 0 <= codes[n,l] < rvq_k, U has orthonormal columns, and for the
 *    Newton-Schulz retraction sigma_max(U - lr xi) < sqrt(3) (S11).
 *  - There is no CPU fallback: without a CUDA device every compute call returns MAPL_ERR_CUDA.
 */
#ifndef MAPL_H_
#define MAPL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  MAPL_OK = 0,
  MAPL_ERR_INVALID_ARG = -1,   /* NULL required pointer, non-positive size, inconsistent combination */
  MAPL_ERR_UNSUPPORTED = -2,   /* valid request outside the implemented envelope (see each call)     */
  MAPL_ERR_ALIGNMENT = -3,     /* a device pointer is not 16-byte aligned                             */
  MAPL_ERR_WORKSPACE = -4,     /* workspace NULL or smaller than mapl_*_workspace_bytes()             */
  MAPL_ERR_CUDA = -5           /* CUDA runtime error (no device, launch failure)                      */
} mapl_status;

typedef enum { MAPL_F32 = 0, MAPL_BF16 = 1 } mapl_dtype;
typedef enum { MAPL_RETRACT_QR = 0, MAPL_RETRACT_NS = 1 } mapl_retraction;

/* One stage boundary (activation X^{b_p} in R^{B x T x d}, N = B*T tokens). */
typedef struct {
  int64_t n_tokens;      /* N >= 0 (N == 0: the call is a no-op apart from zeroing overwrite outputs) */
  int32_t d;             /* hidden size; d >= 8, d % 8 == 0                                          */
  int32_t r;             /* projector rank; 8 <= r <= d, r % 8 == 0; U is [d,r]                      */
  int32_t act_dtype;     /* mapl_dtype of H, Hhat, g, dH, Z, gz                                      */
  int32_t rvq_levels;    /* L; 0 = RVQ off; L <= 8                                                   */
  int32_t rvq_k;         /* K codewords per level (>= 1 when L > 0); codebooks are [L,K,r] fp32       */
  int32_t rvq_group_dim; /* must be r or 0 (one group: full-vector RVQ, S3); grouped MCVQ = next     */
  int32_t vocab;         /* V; A is [V,ra]                                                           */
  int32_t anchor_rank;   /* ra; 0 = no anchor term; else ra % 8 == 0; B is [ra,d]                    */
  const void* param_pack; /* optional DEVICE pointer to the prepared parameter pack written by
                            mapl_pack_params() for these U, B, codebooks (mapl_param_pack_bytes() bytes);
                            NULL = every call re-derives what it needs in its workspace.  The caller
                            guarantees the pack is current (re-pack after every parameter update).   */
} mapl_boundary_desc;

/* Static strings for a status code / the library build ("mapl-b200 x.y sm_100a"). */
const char* mapl_status_string(int status);
const char* mapl_version(void);
/* cudaError_t of the most recent MAPL_ERR_CUDA on the calling thread (0 if none). */
int mapl_last_cuda_error(void);

/* Device scratch the three codec calls need for `desc` (max over the three), in bytes; 0 on an
 * invalid descriptor.  The same workspace may be reused by consecutive calls on one stream.     */
size_t mapl_workspace_bytes(const mapl_boundary_desc* desc);
/* Device scratch for mapl_stiefel_step on `batch` projectors of shape [d,r].                    */
size_t mapl_stiefel_workspace_bytes(int32_t d, int32_t r, int32_t batch);

/* PARAMETER PACK (optional).  The tensor-core kernels read U, B and the codebooks as bf16 operand
 * tiles (U additionally as a two-term bf16 split when RVQ follows, so z stays fp32-accurate; the
 * codebooks as fp16 scaled per level by a power of two) plus per-codeword half squared norms.  mapl_pack_params writes that derived copy into caller-owned
 * device memory `pack_out` (mapl_param_pack_bytes(desc) bytes, 256-byte aligned; 0 bytes when the
 * boundary runs on the fp32 kernels: then pack_out may be NULL and the call is a no-op).  In the
 * paper's schedule the parameters change once per optimizer step while ~128 micro-batches cross
 * the boundary, so the pack is made once per step and referenced from
 * desc.param_pack.  B / codebooks may be NULL when anchor_rank / rvq_levels is 0.  Otherwise a
 * NULL B or NULL codebooks leaves that section of an existing pack as it is: after a projector
 * update (mapl_stiefel_step) call it with U alone, since B and the codebooks did not change.  The
 * first pack of a buffer must pass everything the descriptor uses.                                */
size_t mapl_param_pack_bytes(const mapl_boundary_desc* desc);
int mapl_pack_params(const mapl_boundary_desc* desc, const float* U, const float* B, const float* codebooks,
                     void* pack_out, void* cuda_stream);

/* ENCODE (sender side).  P:73 Eq. 1 with h already centred (S6): z_n = U^T h_n.
 * If desc.rvq_levels == L > 0 (S3, S4): rho_0 = z_n; for l < L:
 *   codes[n,l] = argmin_k || rho_l - C[l,k,:] ||^2 (lowest k on ties), rho_{l+1} = rho_l - C[l,codes[n,l],:].
 * z stays on chip between levels.
 *   H          [N,d] act dtype, read-only.
 *   U          [d,r] fp32.
 *   codebooks  [L,K,r] fp32 (ignored / may be NULL when L == 0).
 *   Zq_out     [N,r] act dtype.  L == 0: required, receives z (the wire payload, 2r bytes/token in
 *              bf16).  L > 0: optional, receives zhat_n = sum_l C[l,codes[n,l],:].
 *   codes_out  [N,L] int32; required when L > 0.
 * Unsupported: rvq_group_dim not in {0, r}; L > 0 with r > 512.                                */
int mapl_encode(const mapl_boundary_desc* desc, const void* H, const float* U, const float* codebooks,
                void* Zq_out, int32_t* codes_out, void* workspace, size_t workspace_bytes,
                void* cuda_stream);

/* ENCODE WITH RVQ, NO WORKSPACE AND NO ALLOCATION (csrc/static_scratch.cu).  For callers that cannot allocate device
 * memory and so cannot give mapl_encode a workspace (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc).  Same operation and arguments as mapl_encode with desc.rvq_levels >= 1 (S3, S4), run on
 * the fp32 SIMT kernels whatever the shape (the kernels mapl_encode uses for fp32 activations and for shapes outside the
 * tensor-core envelope): its results are those of that path.  Its one piece of scratch, the half squared norms of the
 * codewords ([L*K] fp32), lives in a device array inside the library: mapl_static_scratch_rows() floats (16384 = 64 KB,
 * held by every GPU that loads the library until the process exits).
 *   desc.rvq_levels * desc.rvq_k > mapl_static_scratch_rows()  ->  MAPL_ERR_WORKSPACE, nothing is launched.
 *   desc.rvq_levels == 0 -> MAPL_ERR_INVALID_ARG (there is no scratch to speak of: use mapl_encode).
 *   desc.param_pack is ignored.  Other arguments, layouts and errors: as mapl_encode.
 * The call and everything under it call no cudaMalloc / cudaFree / allocating library routine (with
 * mapl_profile_enable(0), the default: launch timing creates CUDA events).  The first call on each device looks the
 * array's address up (cudaGetSymbolAddress): make one call per device before capturing a graph.
 * All calls on a device share the array.  A call overwrites the L*K entries it uses before reading them and nothing
 * has to start at zero, so calls in stream order are independent of each other; calls that can OVERLAP on the GPU
 * (different streams, concurrent graph branches) race on the array: the caller serialises them.                  */
size_t mapl_static_scratch_rows(void);
int mapl_encode_rvq_static(const mapl_boundary_desc* desc, const void* H, const float* U, const float* codebooks,
                           void* Zq_out, int32_t* codes_out, void* cuda_stream);

/* DECODE (receiver side).  P:75 Eq. 2 + P:106 Eq. 3: hhat_n = U zhat_n + B^T A[tok_n,:].
 *   Z / codes  exactly one non-NULL.  Z [N,r] act dtype is used as zhat; codes [N,L] int32 are
 *              dequantised (zhat_n = sum_l C[l,codes[n,l],:], needs L > 0 and codebooks).
 *   tok, A, B  required when desc.anchor_rank > 0 (only token ids cross the wire).
 *   Hhat_out   [N,d] act dtype.                                                                 */
int mapl_decode(const mapl_boundary_desc* desc, const void* Z, const int32_t* codes, const float* U,
                const float* codebooks, const int32_t* tok, const float* A, const float* B,
                void* Hhat_out, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* BACKWARD of loss(Hhat) through decode and encode, straight-through across the quantiser (S7).
 * With g = dL/dHhat [N,d] ("route the gradient through the same orthogonal projector"):
 *   gz   = g U                                   [N,r] act dtype (what crosses the wire backwards)
 *   dU   = g^T Zhat (+ H^T gz when H != NULL)    [d,r] fp32   (Alg. 1 l.4, S8)
 *   dA[v,:] = sum_{n: tok_n = v} B g_n           [V,ra] fp32  (E_small is trainable)
 *   dB   = A[tok]^T g                            [ra,d] fp32  (P_p is frozen in the paper: optional)
 *   dH   = gz U^T                                [N,d] act dtype (optional; needs H != NULL)
 *   Z / codes  exactly one non-NULL: the zhat the forward pass decoded (as in mapl_decode).
 *   H          may be NULL: only the decode-side term of dU is formed and dH_out must be NULL.
 *   gz_out, dU_out required.  dA_out required when anchor_rank > 0 unless A, B, tok are all NULL
 *   (anchor ignored).  dB_out, dH_out optional (NULL = skipped).
 *   accumulate 0: dU, dA, dB are overwritten (rows of dA for absent tokens become 0);
 *              1: results are added to their current contents (micro-batch accumulation).       */
int mapl_codec_backward(const mapl_boundary_desc* desc, const void* g_Hhat, const void* H, const void* Z,
                        const int32_t* codes, const float* U, const float* codebooks, const int32_t* tok,
                        const float* A, const float* B, void* gz_out, float* dU_out, float* dA_out,
                        float* dB_out, void* dH_out, int accumulate, void* workspace,
                        size_t workspace_bytes, void* cuda_stream);

/* SENDER-SIDE ANCHOR CENTRING (Eq. 1 in full; SURVEY 8f "next" row 1, reading S6).  The hot path
 * takes h as the already centred residual; these two calls add the subtraction of the sender's own
 * factorised anchor (Eq. 3):
 *     z = U^T (h - A_s[tok] B_s)  =  U^T h - T[tok],      T = A_s (B_s U)   [V,r] fp32.
 * mapl_center_table forms T once per parameter update (two small fp32 GEMMs; `workspace` of
 * mapl_center_workspace_bytes(desc) bytes holds B_s U); mapl_encode_centered is mapl_encode with the row
 * T[tok_n] subtracted from the fp32 accumulator of token n before anything is rounded or quantised, so
 * the RVQ codes are those of the centred z.  Arguments as mapl_encode, plus tok [N] int32 (0 <= tok < V)
 * and center_table [V,r] fp32.  A_s [V,ra], B_s [ra,d] (the sender's anchor factors; desc.vocab and
 * desc.anchor_rank describe them).
 * mapl_center_backward is the backward of the centring term for gz = dL/dz ([N,r], activation dtype: the gz_out
 * of mapl_codec_backward):  with D[v,:] = sum_{n: tok_n = v} gz_n and Q = A_s^T D,
 *     dA_s = - D (B_s U)^T   [V,ra];    dB_s = - Q U^T   [ra,d] (optional, NULL = skipped);
 *     dU  += - B_s^T Q       [d,r]      (always ADDED: it completes the H^T gz that mapl_codec_backward formed
 *                                        with the uncentred H to (H - A_s[tok] B_s)^T gz).
 * accumulate 0 / 1 applies to dA_s and dB_s as in mapl_codec_backward.  fp32 arithmetic; work is O(V r ra),
 * independent of N apart from the scatter.  workspace: mapl_center_backward_workspace_bytes(desc).   */
size_t mapl_center_workspace_bytes(const mapl_boundary_desc* desc);
size_t mapl_center_backward_workspace_bytes(const mapl_boundary_desc* desc);
int mapl_center_table(const mapl_boundary_desc* desc, const float* A_s, const float* B_s, const float* U,
                      float* table_out, void* workspace, size_t workspace_bytes, void* cuda_stream);
int mapl_encode_centered(const mapl_boundary_desc* desc, const void* H, const int32_t* tok, const float* center_table,
                         const float* U, const float* codebooks, void* Zq_out, int32_t* codes_out, void* workspace,
                         size_t workspace_bytes, void* cuda_stream);
int mapl_center_backward(const mapl_boundary_desc* desc, const void* gz, const int32_t* tok, const float* A_s,
                         const float* B_s, const float* U, float* dA_s_out, float* dB_s_out, float* dU_inout,
                         int accumulate, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* STIEFEL STEP on `batch` independent projectors, U_inout and G strided [batch,d,r] fp32.
 *   S = U^T G;  xi = G - U (S + S^T)/2 (Eq. 4);  Y = U - lr xi;
 *   MAPL_RETRACT_QR: U <- Q of the thin QR of Y with diag(R) > 0 (unique, S17);
 *   MAPL_RETRACT_NS: X_0 = Y, X_{j+1} = X_j (3I - X_j^T X_j)/2, U <- X_{ns_iters} (S11; the
 *                    reported configuration is ns_iters = 5; 1 <= ns_iters <= 16).
 *   U_inout is updated in place.  fp32 storage, fp32-accurate arithmetic: ||U^T U - I||_F <= 1e-5
 *   after the call for inputs in the documented regime.  (With d % 128 == 0, r % 128 == 0,
 *   r >= 256 the [d,r]-sized products run on the tensor cores as exact three-plane bf16 splits,
 *   six MMAs per product; otherwise fp32 FFMA kernels.  QR: CholeskyQR2 in fp32 -- blocked
 *   Cholesky of the Gram matrix and a blocked triangular inverse, twice; it needs cond(Y) well
 *   below 1e3, which holds for a step from an orthonormal U.  Measured residuals: <= 5e-6 on the
 *   tensor-core shapes up to r = 1024; the FFMA kernels stay below 1e-5 for r <= 768 at
 *   d <= 2048 and reach 1.1e-5 at d = r = 1024 -- plain fp32 sums over d.)
 *   info_out   optional device [batch,2] fp32: ||xi||_F and ||U^T U - I||_F after the update.
 * Requires 8 <= r <= d, r % 8 == 0, d % 8 == 0, r <= 1024.                                      */
int mapl_stiefel_step(int32_t d, int32_t r, int32_t batch, float* U_inout, const float* G, float lr,
                      int32_t retraction, int32_t ns_iters, float* info_out, void* workspace,
                      size_t workspace_bytes, void* cuda_stream);

/* LAUNCH ACCOUNTING (diagnostics; host-side state, not thread-safe).  Every kernel (and memset)
 * the library enqueues is counted per kernel id.  With timing switched on each launch is also
 * bracketed by a CUDA-event pair on its own stream; mapl_profile_read() synchronises on those
 * events.  Do not switch timing on while a stream is being captured into a CUDA graph.
 *   mapl_profile_kernel_count()      number of kernel ids
 *   mapl_profile_kernel_name(kid)    static name of kernel id `kid` ("" if out of range)
 *   mapl_profile_enable(on)          1: time launches from now on; 0: stop (counting never stops)
 *   mapl_profile_reset()             zero all counters and timers
 *   mapl_profile_read(kid, ...)      launches since reset, launches that were timed, their total ms
 *                                    (any out pointer may be NULL)                                  */
int mapl_profile_kernel_count(void);
const char* mapl_profile_kernel_name(int kid);
void mapl_profile_enable(int timing_on);
void mapl_profile_reset(void);
int mapl_profile_read(int kid, long long* launches, long long* timed_launches, double* total_ms);

/* GROUPED MULTI-CODEBOOK VQ of a wire payload (Sec. 3.5; reading S3; SURVEY 8f "next" row 3).
 * X [N,r] in the activation dtype is a stored payload: the Z written by mapl_encode (RVQ off) or the gz written by
 * mapl_codec_backward.  Its r channels are cut into r/2 groups of G = 2 consecutive channels; group g is residual-
 * vector-quantised on its own over `levels` rounds with the 2-d codewords codebooks[l, k, 2g:2g+2] (codebooks
 * [levels,k,r] fp32, the layout of the full-vector RVQ), squared Euclidean distance, lowest index on ties (S4).
 *   codes_out [N, levels, r/2] uint8 (k <= 256): (r/2) levels bytes per token -- 256 B at r = 256, levels = 2.
 *   Xq_out    optional [N,r] activation dtype: the dequantised payload (sum of the chosen codewords, rounded once).
 * mapl_mcvq_dequantize rebuilds Xq from the codes on the receiving side (feed it to mapl_decode as Z, or use it as
 * gz).  r % 8 == 0, 1 <= levels <= 4.  No workspace.                                                            */
int mapl_mcvq_quantize(int64_t n_tokens, int32_t r, int32_t act_dtype, int32_t levels, int32_t k, const void* X,
                       const float* codebooks, uint8_t* codes_out, void* Xq_out, void* cuda_stream);
int mapl_mcvq_dequantize(int64_t n_tokens, int32_t r, int32_t act_dtype, int32_t levels, int32_t k, const uint8_t* codes,
                         const float* codebooks, void* Xq_out, void* cuda_stream);

/* STREAMING CODEBOOK SYNCHRONISATION, device side, and the retained-energy diagnostic (SURVEY 8f "next" row 4).
 * P:151-153 / P:405-411: sender and receiver keep identical codebooks by shipping a random subset of the codewords
 * with every micro-batch instead of the whole table.  The codebooks are viewed as a table [L*K, r] fp32:
 *   mapl_codebook_delta_pack   rows_out[i,:] = codebooks[idx[i],:]   (sender: the m rows this micro-batch carries)
 *   mapl_codebook_delta_apply  codebooks[idx[i],:] = rows[i,:]       (receiver: patch its copy; idx without duplicates)
 * idx [m] int32 device, flat row numbers in [0, L*K).  WHICH rows travel when is host protocol logic (reading S15: a
 * seeded permutation of the rows cut into `interval` = 5 parts, part t mod 5 with micro-batch t: after 5 micro-batches
 * every row has been refreshed).  r % 4 == 0.
 *   mapl_energy_retained   sums_inout[0] += ||Z||_F^2, sums_inout[1] += ||H||_F^2  (device double[2], caller-zeroed):
 *   E = sums[0] / sums[1] is the energy of the activations retained under projection, ||X A||_F^2 / ||X||_F^2 of
 *   Fig. 4(b).  H [N,d], Z [N,r] in the activation dtype (Z as written by mapl_encode, RVQ off).          */
int mapl_codebook_delta_pack(const float* codebooks, int32_t r, const int32_t* idx, int32_t m, float* rows_out,
                             void* cuda_stream);
int mapl_codebook_delta_apply(float* codebooks_inout, int32_t r, const int32_t* idx, int32_t m, const float* rows,
                              void* cuda_stream);
int mapl_energy_retained(int64_t n_tokens, int32_t d, int32_t r, int32_t act_dtype, const void* H, const void* Z,
                         double* sums_inout, void* cuda_stream);

/* FULL SPEL STEP (Eq. 4-7; SURVEY 8f "next" row 2) on `batch` projectors, U, G, M strided [batch,d,r] fp32:
 *     xi = G - U sym(U^T G)                      (Eq. 4, tangent projection)
 *     m  <- beta m + (1 - beta) xi               (Eq. 5, heavy-ball momentum; M_inout updated in place)
 *     d  = NS_{lmo_iters}( m / ||m||_F )         (Eq. 6, spectral LMO direction)
 *     U  <- NS_{retr_iters}( U - lr d )          (Eq. 7, retraction)
 * The paper's PolarExpress [2] is not printed in it; here both polar steps are the cubic Newton-Schulz iteration
 * X <- X (3I - X^T X)/2 (reading S11), for Eq. 6 from the Frobenius-normalised momentum (all singular values <= 1; with
 * the paper's 5 iterations the small ones are only partly lifted towards 1, as in Muon), for Eq. 7 with the paper's 7.
 * ||m||_F == 0 gives d = 0.  1 <= lmo_iters, retr_iters <= 16; 0 <= beta <= 1.  Same shapes, arithmetic paths and
 * workspace as mapl_stiefel_step (mapl_spel_workspace_bytes).                                                        */
size_t mapl_spel_workspace_bytes(int32_t d, int32_t r, int32_t batch);
int mapl_spel_step(int32_t d, int32_t r, int32_t batch, float* U_inout, const float* G, float* M_inout, float lr,
                   float beta, int32_t lmo_iters, int32_t retr_iters, void* workspace, size_t workspace_bytes,
                   void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* MAPL_H_ */
