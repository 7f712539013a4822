// stiefel.cu -- mapl_stiefel_step: tangent projection (Eq. 4), step, and retraction
// onto St(d,r) by thin QR (CholeskyQR2, diag(R) > 0) or by a fixed number of cubic Newton-Schulz
// polar iterations (count passed in; 5 in every reported number).  fp32 storage and fp32-accurate
// arithmetic throughout: tcgen05 has no fp32 kind and a single TF32 pass cannot hold
// ||U^T U - I||_F <= 1e-5, so the products are fp32 FFMA kernels here or,
// for d, r multiples of 128 and r >= 256, exact three-plane bf16 splits on the tensor cores (tc_stiefel.cu).
//
//   Y = U - lr (G - U sym(U^T G)) = U (I + lr sym(S)) - lr G,   S = U^T G
#include "common.cuh"
#include <stdlib.h>

#include "profile.cuh"
#include "tc_stiefel.cuh"

namespace mapl {
namespace {

constexpr int NB = 32;

__global__ void k_step_matrix(const float* __restrict__ S, float* __restrict__ M1, int r, float lr) {
  // M1 = I + lr (S + S^T)/2, batched over blockIdx.y
  const long long off = (long long)blockIdx.y * r * r;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= r * r) return;
  const int a = idx / r, b = idx % r;
  M1[off + idx] = (a == b ? 1.f : 0.f) + lr * 0.5f * (S[off + a * r + b] + S[off + b * r + a]);
}

// element (a,b) of a symmetric [r,r] matrix of which only the 64x64 tiles on or above the diagonal are stored
__device__ __forceinline__ float sym_at(const float* __restrict__ G, int r, int a, int b) {
  return (a / 64 <= b / 64) ? G[(long long)a * r + b] : G[(long long)b * r + a];
}

__global__ void k_ns_poly(const float* __restrict__ Gm, float* __restrict__ M, int r) {
  // M = (3I - Gm)/2, Gm = X^T X stored as upper tiles
  const long long off = (long long)blockIdx.y * r * r;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= r * r) return;
  const int a = idx / r, b = idx % r;
  M[off + idx] = 0.5f * ((a == b ? 3.f : 0.f) - sym_at(Gm + off, r, a, b));
}

// out[b*2 + slot] = sqrt(sum_i (scale*(X[i] - Yv[i]))^2)   (Yv may be null: then X - I on an [r,r] matrix)
__global__ void k_fro_norm(const float* __restrict__ X, const float* __restrict__ Yv, float scale, long long n,
                           int r_if_identity, float* __restrict__ out, int slot) {
  __shared__ float red[32];
  const long long off = (long long)blockIdx.x * n;
  float s = 0.f;
  for (long long i = threadIdx.x; i < n; i += blockDim.x) {
    float v;
    if (Yv) v = scale * (X[off + i] - Yv[off + i]);
    else {
      const int a = (int)(i / r_if_identity), b = (int)(i % r_if_identity);
      v = X[off + i] - (a == b ? 1.f : 0.f);
    }
    s = fmaf(v, v, s);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x % 32 == 0) red[threadIdx.x / 32] = s;
  __syncthreads();
  if (threadIdx.x < 32) {
    s = threadIdx.x < blockDim.x / 32 ? red[threadIdx.x] : 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0) out[blockIdx.x * 2 + slot] = sqrtf(s);
  }
}

// ---------------------------------------------------------------- blocked upper Cholesky G = R^T R with look-ahead
// Right-looking, NB = 32 columns per panel, ONE launch per panel (k_chol_step).  A panel's diagonal block D is
// factored by the launch BEFORE the one that uses it: the CTA that updates the leading trailing tile factors the
// next diagonal block from its own result (look-ahead).  The panel rows D^-T G[p:p+NB, cols] are a forward
// substitution (one thread per column) that every CTA redoes for the two column ranges its tile needs, instead of a
// single CTA solving the whole panel.  The critical path of a launch is load -> solve -> update -> factor; the
// inverses of the diagonal blocks (seed of the blocked triangular inverse below) are computed off that path by one
// extra CTA per launch and land in the diagonal blocks of Xinv.

// warp-level: factor the NB x NB block in Dn (upper triangle read; rows / columns past nb padded with the identity),
// write R (strict lower part zeroed) to Gd (pitch r).  lane = column.
__device__ __forceinline__ void diag_factor(float (*Dn)[NB + 1], int nb, float* __restrict__ Gd, int r, int lane) {
  float col[NB];                     // col[a] = D[a][lane]; row j is exchanged by shuffles
#pragma unroll
  for (int a = 0; a < NB; ++a) col[a] = (a < nb && lane < nb) ? Dn[a][lane] : (a == lane ? 1.f : 0.f);
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    const float c = __shfl_sync(0xffffffffu, col[j], j);
    float y = rsqrtf(c);
    y = y * fmaf(-0.5f * c * y, y, 1.5f);                                      // one Newton step: 1/sqrt(c) to ~1 ulp
    const float rowj = lane == j ? c * y : (lane > j ? col[j] * y : col[j]);   // R[j][lane]
    col[j] = rowj;
#pragma unroll
    for (int a = j + 1; a < NB; ++a) {
      const float dja = __shfl_sync(0xffffffffu, rowj, a);                      // R[j][a]
      if (a <= lane) col[a] = fmaf(-dja, rowj, col[a]);
    }
  }
#pragma unroll
  for (int a = 0; a < NB; ++a)
    if (a < nb && lane < nb) Gd[(long long)a * r + lane] = a <= lane ? col[a] : 0.f;
}

// warp-level: Xd = R^-1 for the upper-triangular block in Dn (padded with the identity past nb).  lane = column:
// back substitution with x[k] = 0 for k > lane, so the loops are uniform and every Dn read is a broadcast.
__device__ __forceinline__ void diag_invert(float (*Dn)[NB + 1], int nb, float* __restrict__ Xd, int r, int lane) {
  float x[NB];
#pragma unroll
  for (int a = NB - 1; a >= 0; --a) {
    float s = a == lane ? 1.f : 0.f;
#pragma unroll
    for (int k = a + 1; k < NB; ++k) s = fmaf(-Dn[a][k], x[k], s);
    x[a] = a <= lane ? s / Dn[a][a] : 0.f;
  }
#pragma unroll
  for (int a = 0; a < NB; ++a)
    if (a < nb && lane < nb) Xd[(long long)a * r + lane] = x[a];
}

// first diagonal block (one warp per batch item)
__global__ void __launch_bounds__(32) k_chol_first(float* __restrict__ Gb, int r) {
  __shared__ float Dn[NB][NB + 1];
  float* G = Gb + (long long)blockIdx.x * r * r;
  const int lane = threadIdx.x, nb = min(NB, r);
  for (int a = 0; a < nb; ++a) Dn[a][lane] = lane < nb ? G[(long long)a * r + lane] : 0.f;
  __syncwarp();
  diag_factor(Dn, nb, G, r, lane);
}

// Panel p (diagonal block already factored); q = p + NB.  grid = (64x64 tiles on or above the diagonal of the trailing
// block G[q:, q:]  +  1, batch).  Tile CTAs: P = D^-T G[p:p+NB, cols] for the tile's row range and column range,
// tile -= P_r^T P_c; diagonal tiles store P (= rows p..p+NB of R) into the SEPARATE matrix Pb (other CTAs of the
// launch still read the raw panel rows of G); tile (0,0) then factors the next diagonal block.  The extra CTA inverts
// D into Xinv[p:p+NB, p:p+NB].  R is thus held in two matrices: its diagonal NB-blocks in G, the rest in Pb.
__global__ void __launch_bounds__(256) k_chol_step(float* __restrict__ Gb, float* __restrict__ Xb, float* __restrict__ Pb, int r, int p) {
  constexpr int TS = 64, PAD = 4;
  __shared__ float Di[NB][NB + 1];
  __shared__ float rd[NB];
  __shared__ __align__(16) float Pr[NB][TS + PAD], Pc[NB][TS + PAD];
  float* G = Gb + (long long)blockIdx.y * r * r;
  float* X = Xb + (long long)blockIdx.y * r * r;
  float* P = Pb + (long long)blockIdx.y * r * r;
  const int t = threadIdx.x, q = p + NB, nt = q < r ? (r - q + TS - 1) / TS : 0;
  if ((int)blockIdx.x == nt * (nt + 1) / 2) {                 // the inverse CTA
    if (t < 32) {
      const int nb = min(NB, r - p);
      for (int a = 0; a < NB; ++a) Di[a][t] = (a < nb && t < nb) ? G[(long long)(p + a) * r + p + t] : (a == t ? 1.f : 0.f);
      __syncwarp();
      diag_invert(Di, nb, X + (long long)p * r + p, r, t);
    }
    return;
  }
  int rem = blockIdx.x, tm = 0;
  while (rem >= nt - tm) { rem -= nt - tm; ++tm; }
  const int tn = tm + rem, m0 = q + tm * TS, n0 = q + tn * TS;
  for (int i = t; i < NB * NB; i += 256) Di[i / NB][i % NB] = G[(long long)(p + i / NB) * r + p + i % NB];
  // raw panel rows over the tile's row range (-> Pr) and column range (-> Pc)
  for (int i = t; i < NB * TS / 4; i += 256) {
    const int j = i / (TS / 4), c = (i % (TS / 4)) * 4;
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    *reinterpret_cast<float4*>(&Pr[j][c]) = m0 + c < r ? *reinterpret_cast<const float4*>(G + (long long)(p + j) * r + m0 + c) : z;
    *reinterpret_cast<float4*>(&Pc[j][c]) = n0 + c < r ? *reinterpret_cast<const float4*>(G + (long long)(p + j) * r + n0 + c) : z;
  }
  // this thread's part of the trailing tile, in flight during the solve
  const int tx = t % 16, ty = t / 16;
  float4 tv[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i, n = n0 + tx * 4;
    tv[i] = (m < r && n < r) ? *reinterpret_cast<const float4*>(G + (long long)m * r + n) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();
  if (t < NB) rd[t] = 1.f / Di[t][t];
  __syncthreads();
  if (t < 2 * TS) {   // forward substitution D^T x = g, in place: thread = one column of Pr (t < 64) or Pc
    float (*Pm)[TS + PAD] = t < TS ? Pr : Pc;
    const int c = t % TS;
    float x[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      float sacc = Pm[j][c];
#pragma unroll
      for (int k = 0; k < j; ++k) sacc = fmaf(-Di[k][j], x[k], sacc);
      x[j] = sacc * rd[j];
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) Pm[j][c] = x[j];
    if (t >= TS && tm == tn && n0 + c < r) {
#pragma unroll
      for (int j = 0; j < NB; ++j) P[(long long)(p + j) * r + n0 + c] = x[j];
    }
  }
  __syncthreads();
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
#pragma unroll 8
  for (int k = 0; k < NB; ++k) {
    const float4 a = *reinterpret_cast<const float4*>(&Pr[k][ty * 4]);
    const float4 b = *reinterpret_cast<const float4*>(&Pc[k][tx * 4]);
    const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
  }
  const bool lead = tm == 0 && tn == 0;
  float (*Dn)[NB + 1] = Di;                       // the next diagonal block reuses Di (every thread is past the solve)
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i, n = n0 + tx * 4;
    if (m >= r || n >= r) continue;
    float4 v = tv[i];
    v.x -= acc[i][0]; v.y -= acc[i][1]; v.z -= acc[i][2]; v.w -= acc[i][3];
    *reinterpret_cast<float4*>(G + (long long)m * r + n) = v;
    if (lead && ty * 4 + i < NB && tx * 4 < NB) {
      Dn[ty * 4 + i][tx * 4] = v.x; Dn[ty * 4 + i][tx * 4 + 1] = v.y; Dn[ty * 4 + i][tx * 4 + 2] = v.z; Dn[ty * 4 + i][tx * 4 + 3] = v.w;
    }
  }
  if (lead) {
    __syncthreads();
    if (t < 32) diag_factor(Dn, min(NB, r - q), G + (long long)q * r + q, r, t);
  }
}

// One half of a level of the blocked triangular inverse: block size b, pair j covers [o, o+2b), o = 2 b j.
//   phase 0:  T12 = R12 X22      phase 1:  X12 = -X11 T12       (all [r,r] row-major, pitch r)
// grid = (64x64 tiles of a [b,b] block, pairs, batch)
__global__ void __launch_bounds__(256) k_tri_level(const float* __restrict__ Rb, float* __restrict__ Xb, float* __restrict__ Tb,
                                                   int r, int b, int phase) {
  constexpr int TS = 64, KS = 16, PAD = 4;
  __shared__ __align__(16) float As[KS][TS + PAD], Bs[KS][TS + PAD];
  const long long off = (long long)blockIdx.z * r * r;
  const int o = 2 * b * blockIdx.y, o2 = o + b;
  const int M = b, N = min(b, r - o2), K = phase == 0 ? N : M;
  const int tiles_n = (b + TS - 1) / TS;
  const int m0 = (blockIdx.x / tiles_n) * TS, n0 = (blockIdx.x % tiles_n) * TS;
  if (n0 >= N) return;
  const float* A = (phase == 0 ? Rb + off + (long long)o * r + o2 : Xb + off + (long long)o * r + o);
  const float* B = (phase == 0 ? Xb + off + (long long)o2 * r + o2 : Tb + off + (long long)o * r + o2);
  float* C = (phase == 0 ? Tb : Xb) + off + (long long)o * r + o2;
  const int t = threadIdx.x, tx = t % 16, ty = t / 16;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int k0 = 0; k0 < K; k0 += KS) {
    {   // A tile [TS][KS]: row m, 4 consecutive k (stored transposed);  B tile [KS][TS]: row k, 4 consecutive n
      const int m = m0 + t / (KS / 4), k = k0 + (t % (KS / 4)) * 4;
      const float4 a = (m < M && k < K) ? *reinterpret_cast<const float4*>(A + (long long)m * r + k) : z;
      const int ml = t / (KS / 4), kl = (t % (KS / 4)) * 4;
      As[kl][ml] = a.x; As[kl + 1][ml] = a.y; As[kl + 2][ml] = a.z; As[kl + 3][ml] = a.w;
      const int kb = k0 + t / (TS / 4), n = n0 + (t % (TS / 4)) * 4;
      *reinterpret_cast<float4*>(&Bs[t / (TS / 4)][(t % (TS / 4)) * 4]) =
          (kb < K && n < N) ? *reinterpret_cast<const float4*>(B + (long long)kb * r + n) : z;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < KS; ++k) {
      const float4 a = *reinterpret_cast<const float4*>(&As[k][ty * 4]);
      const float4 bb = *reinterpret_cast<const float4*>(&Bs[k][tx * 4]);
      const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {bb.x, bb.y, bb.z, bb.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }
  const float sgn = phase == 0 ? 1.f : -1.f;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i, n = n0 + tx * 4;
    if (m >= M || n >= N) continue;
    *reinterpret_cast<float4*>(C + (long long)m * r + n) = make_float4(sgn * acc[i][0], sgn * acc[i][1], sgn * acc[i][2], sgn * acc[i][3]);
  }
}

struct StWs {
  size_t S, M, Rinv, Rinv2, X0, X1, X2, norm2, Prow, Ptr, Ptr2, Pm, total;   // P*: bf16 planes of the tensor-core path
};
StWs st_carve(int d, int r, int batch) {
  StWs w;
  size_t off = 0;
  auto seg = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  w.S = seg((size_t)batch * r * r * 4);
  w.M = seg((size_t)batch * r * r * 4);
  w.Rinv = seg((size_t)batch * r * r * 4);
  w.Rinv2 = seg((size_t)batch * r * r * 4);
  w.X0 = seg((size_t)batch * d * r * 4);
  w.X1 = seg((size_t)batch * d * r * 4);
  w.X2 = seg((size_t)batch * d * r * 4);          // mapl_spel_step: the LMO direction
  w.norm2 = seg((size_t)batch * 4);
  const bool tcp = tc_st_ok(d, r);
  w.Prow = seg(tcp ? tc_st_plane_bytes(d, r, batch) : 0);
  w.Ptr = seg(tcp ? tc_st_plane_bytes(d, r, batch) : 0);
  w.Ptr2 = seg(tcp ? tc_st_plane_bytes(d, r, batch) : 0);
  w.Pm = seg(tcp ? tc_st_plane_bytes(r, r, batch) : 0);
  w.total = off + 256;
  return w;
}

// ---------------------------------------------------------------- fp32 FFMA GEMMs of the step
// 128x64 output tile, BK = 16, 256 threads x (8x4), register-prefetched double buffering, 128-bit
// global and shared accesses.  Two shapes:
//   kGram : C[r,r] (+)= X[k0:k1, :]^T Y[k0:k1, :]   X, Y row-major [d,r]; split over d, vector reds
//   !kGram: C[d,r]  = alpha A[d,r] M[r,r] (+ beta E)  A row-major (k contiguous), M row-major
// Sizes need only r % 4 == 0 (the ABI asks r % 8 == 0); edges are zero-filled / guarded.
#ifndef MAPL_ST_TM
#define MAPL_ST_TM 64
#endif
#ifndef MAPL_ST_TK
#define MAPL_ST_TK 16
#endif
constexpr int TM = MAPL_ST_TM, TN = 64, TK = MAPL_ST_TK, TPAD = 4;
constexpr int RM = TM / 16;                         // rows per thread (4 or 8); 4 columns per thread
constexpr int LA = TM * TK / 4 / 256, LB = TN * TK / 4 / 256;   // float4 loads per thread per k-step tile

template <bool kGram>
__global__ void __launch_bounds__(256) k_st_gemm(const float* __restrict__ A, const float* __restrict__ B, float* __restrict__ C,
                                                 const float* __restrict__ E, float alpha, float beta, int M, int N, int K, int kper,
                                                 long long sA, long long sB, long long sC, int upper_only,
                                                 int lda, int ldb, int ldc) {      // row pitches (elements) of A, B, C / E
  __shared__ __align__(16) float As[2][TK][TM + TPAD];
  __shared__ __align__(16) float Bs[2][TK][TN + TPAD];
  const int t = threadIdx.x, tx = t % 16, ty = t / 16;      // thread tile: rows ty*RM..+RM-1, cols tx*4..+3
  const int tiles_n = (N + TN - 1) / TN;
  int tm = blockIdx.x / tiles_n, tn = blockIdx.x % tiles_n;
  if (upper_only) {            // symmetric product (TM == TN): blockIdx.x enumerates the tiles with tn >= tm
    int rem = blockIdx.x;
    tm = 0;
    while (rem >= tiles_n - tm) { rem -= tiles_n - tm; ++tm; }
    tn = tm + rem;
  }
  const int m0 = tm * TM, n0 = tn * TN;
  const int kbeg = blockIdx.y * kper, kend = min(K, kbeg + kper);
  A += (long long)blockIdx.z * sA; B += (long long)blockIdx.z * sB; C += (long long)blockIdx.z * sC;
  if (E) E += (long long)blockIdx.z * sC;
  float acc[RM][4];
#pragma unroll
  for (int i = 0; i < RM; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  // one k-step tile (TK rows of k) is fetched into registers while the previous one is multiplied.
  // Measured (ncu): 128x64 tiles or TK = 32 change nothing -- the kernel is limited by occupancy
  // (the step's GEMMs are ~0.3 GFLOP each: 1-3 CTAs per SM) and shared-memory scoreboard stalls.
  float4 ra[LA], rb[LB];
  auto gload = [&](int k0) {
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < LB; ++i) {   // B tile [TK][TN]: row k, 4 consecutive n
      const int f = t + i * 256, k = k0 + f / (TN / 4), n = n0 + (f % (TN / 4)) * 4;
      rb[i] = (k < kend && n < N) ? __ldg(reinterpret_cast<const float4*>(B + (long long)k * ldb + n)) : z;
    }
#pragma unroll
    for (int i = 0; i < LA; ++i) {
      const int f = t + i * 256;
      if (kGram) {   // A tile [TK][TM]: row k, 4 consecutive m
        const int k = k0 + f / (TM / 4), m = m0 + (f % (TM / 4)) * 4;
        ra[i] = (k < kend && m < M) ? __ldg(reinterpret_cast<const float4*>(A + (long long)k * lda + m)) : z;
      } else {       // A tile [TM][TK]: row m, 4 consecutive k
        const int m = m0 + f / (TK / 4), k = k0 + (f % (TK / 4)) * 4;
        ra[i] = (m < M && k < kend) ? __ldg(reinterpret_cast<const float4*>(A + (long long)m * lda + k)) : z;
      }
    }
  };
  auto sstore = [&](int buf) {
#pragma unroll
    for (int i = 0; i < LB; ++i) {
      const int f = t + i * 256;
      *reinterpret_cast<float4*>(&Bs[buf][f / (TN / 4)][(f % (TN / 4)) * 4]) = rb[i];
    }
#pragma unroll
    for (int i = 0; i < LA; ++i) {
      const int f = t + i * 256;
      if (kGram) {
        *reinterpret_cast<float4*>(&As[buf][f / (TM / 4)][(f % (TM / 4)) * 4]) = ra[i];
      } else {
        const int m = f / (TK / 4), k = (f % (TK / 4)) * 4;
        As[buf][k + 0][m] = ra[i].x; As[buf][k + 1][m] = ra[i].y; As[buf][k + 2][m] = ra[i].z; As[buf][k + 3][m] = ra[i].w;
      }
    }
  };
  if (kbeg < kend) {
    gload(kbeg);
    sstore(0);
    __syncthreads();
    int buf = 0;
    for (int k0 = kbeg; k0 < kend; k0 += TK) {
      const bool more = k0 + TK < kend;
      if (more) gload(k0 + TK);
#pragma unroll
      for (int k = 0; k < TK; ++k) {
        float av[RM];
#pragma unroll
        for (int i = 0; i < RM / 4; ++i) {
          const float4 a = *reinterpret_cast<const float4*>(&As[buf][k][ty * RM + 4 * i]);
          av[4 * i] = a.x; av[4 * i + 1] = a.y; av[4 * i + 2] = a.z; av[4 * i + 3] = a.w;
        }
        const float4 bb = *reinterpret_cast<const float4*>(&Bs[buf][k][tx * 4]);
        const float bv[4] = {bb.x, bb.y, bb.z, bb.w};
#pragma unroll
        for (int i = 0; i < RM; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
      }
      if (more) { sstore(buf ^ 1); __syncthreads(); buf ^= 1; }
    }
  }
#pragma unroll
  for (int i = 0; i < RM; ++i) {
    const int m = m0 + ty * RM + i, n = n0 + tx * 4;
    if (m >= M || n >= N) continue;
    float* dst = C + (long long)m * ldc + n;
    if (kGram) {
      asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(alpha * acc[i][0]), "f"(alpha * acc[i][1]),
                   "f"(alpha * acc[i][2]), "f"(alpha * acc[i][3]) : "memory");
    } else {
      float4 v = make_float4(alpha * acc[i][0], alpha * acc[i][1], alpha * acc[i][2], alpha * acc[i][3]);
      if (E) {
        const float4 e = __ldg(reinterpret_cast<const float4*>(E + (long long)m * ldc + n));
        v.x = fmaf(beta, e.x, v.x); v.y = fmaf(beta, e.y, v.y); v.z = fmaf(beta, e.z, v.z); v.w = fmaf(beta, e.w, v.w);
      }
      *reinterpret_cast<float4*>(dst) = v;
    }
  }
}

// Gm[b] = X[b]^T X2[b]  ([r,r], split over d with vector reds).  upper_only (X2 == X, TM == TN): only the
// 64x64 tiles on or above the diagonal are computed; readers use sym_at().
int gram(const float* X, const float* X2, float* Gm, int d, int r, int batch, cudaStream_t st, bool upper_only = false) {
  { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(Gm, 0, (size_t)batch * r * r * 4, st)); }
  const int nt = (r + TN - 1) / TN;
  upper_only = upper_only && TM == TN;
  const int tiles = upper_only ? nt * (nt + 1) / 2 : ((r + TM - 1) / TM) * nt;
  int splits = (2 * 148 + tiles * batch - 1) / (tiles * batch);          // about two waves of CTAs
  int kper = ((d + splits - 1) / splits + TK - 1) / TK * TK;
  if (kper < 4 * TK) kper = 4 * TK;
  splits = (d + kper - 1) / kper;
  KernelScope ks(KID_ST_GEMM, st);
  k_st_gemm<true><<<dim3(tiles, splits, batch), 256, 0, st>>>(X, X2, Gm, nullptr, 1.f, 0.f, r, r, d, kper, (long long)d * r,
                                                            (long long)d * r, (long long)r * r, upper_only ? 1 : 0, r, r, r);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

// C[b] = alpha X[b] M[b] (+ beta E[b]);  X, C, E are [rows, r], M is [r, r]
int right_mul(const float* X, const float* M, float* C, const float* E, float beta, int rows, int r, int batch,
              cudaStream_t st, float alpha = 1.f) {
  const int tiles = ((rows + TM - 1) / TM) * ((r + TN - 1) / TN);
  KernelScope ks(KID_ST_GEMM, st);
  k_st_gemm<false><<<dim3(tiles, 1, batch), 256, 0, st>>>(X, M, C, E, alpha, beta, rows, r, r, r, (long long)rows * r,
                                                         (long long)r * r, (long long)rows * r, 0, r, r, r);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

// Upper Cholesky G = R^T R of `batch` SPD [r,r] matrices (upper triangle read) and Xinv = R^-1.
// Launches: 1 + r/NB for the factorisation (k_chol_first, k_chol_step per panel), then per doubling level b = NB,
// 2 NB, ... two block products (R^-1 of [[R11, R12], [0, R22]] is [[X11, -X11 R12 X22], [0, X22]]): ~r^3/3 flops
// in 2 log2(r/NB) launches.  Rp receives the off-diagonal part of R, T is scratch (all [batch][r][r]).
int chol_inverse_blocked(float* G, float* Xinv, float* Rp, float* T, int r, int batch, cudaStream_t st) {
  { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(Xinv, 0, (size_t)batch * r * r * 4, st)); }
  {
    KernelScope ks(KID_ST_CHOL, st);
    k_chol_first<<<batch, 32, 0, st>>>(G, r);
    MAPL_CUDA_CHECK(cudaGetLastError());
  }
  for (int p = 0; p < r; p += NB) {        // the last launch has no trailing block: only the inverse CTA
    const int nt = p + NB < r ? (r - p - NB + 63) / 64 : 0;
    KernelScope ks(KID_ST_CHOL, st);
    k_chol_step<<<dim3(nt * (nt + 1) / 2 + 1, batch), 256, 0, st>>>(G, Xinv, Rp, r, p);
    MAPL_CUDA_CHECK(cudaGetLastError());
  }
  for (int b = NB; b < r; b *= 2) {
    const int pairs = (r - b + 2 * b - 1) / (2 * b), tiles = ((b + 63) / 64) * ((b + 63) / 64);
    for (int phase = 0; phase < 2; ++phase) {
      KernelScope ks(KID_ST_TRI_INV, st);
      k_tri_level<<<dim3(tiles, pairs, batch), 256, 0, st>>>(Rp, Xinv, T, r, b, phase);
      MAPL_CUDA_CHECK(cudaGetLastError());
    }
  }
  return MAPL_OK;
}

// ---------------------------------------------------------------- full SPEL step (Eq. 4-7)
// M = -(S + S^T)/2 (batched [r,r])
__global__ void k_neg_sym(const float* __restrict__ S, float* __restrict__ M, int r) {
  const long long off = (long long)blockIdx.y * r * r;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= r * r) return;
  const int a = idx / r, b = idx % r;
  M[off + idx] = -0.5f * (S[off + a * r + b] + S[off + b * r + a]);
}

// m <- beta m + (1 - beta) xi ;  norm2[b] += sum m^2   (norm2 zeroed before)
__global__ void __launch_bounds__(256) k_momentum(float* __restrict__ Mom, const float* __restrict__ xi, float beta, long long n,
                                                  float* __restrict__ norm2) {
  __shared__ float red[8];
  const long long off = (long long)blockIdx.y * n;
  float s = 0.f;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
    const float m = fmaf(beta, Mom[off + i], (1.f - beta) * xi[off + i]);
    Mom[off + i] = m;
    s = fmaf(m, m, s);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x % 32 == 0) red[threadIdx.x / 32] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < 8; ++k) s += red[k];
    atomicAdd(norm2 + blockIdx.y, s);
  }
}

// out = a X + c Y / sqrt(norm2[b])   (norm2 == nullptr: plain a X + c Y;  norm2[b] == 0: the Y term is 0)
__global__ void k_axpby_scaled(float* __restrict__ out, const float* __restrict__ X, float a, const float* __restrict__ Y, float c,
                               const float* __restrict__ norm2, long long n) {
  const long long off = (long long)blockIdx.y * n;
  float cs = c;
  if (norm2 != nullptr) { const float q = norm2[blockIdx.y]; cs = q > 0.f ? c / sqrtf(q) : 0.f; }
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    out[off + i] = (X != nullptr ? a * X[off + i] : 0.f) + cs * Y[off + i];
}

struct StCtx {
  int d, r, batch; cudaStream_t st; bool tc;
  float *S, *M;
  __nv_bfloat16 *Prow, *Ptr, *Ptr2, *Pm;
};

// xi = G - U sym(U^T G)  (Eq. 4) into `out`
int ctx_tangent(const StCtx& c, const float* U, const float* G, float* out) {
  const int d = c.d, r = c.r, batch = c.batch;
  if (c.tc) {
    MAPL_RETURN_IF(tc_st_split(U, d, r, batch, 0, 0.f, c.Prow, c.Ptr, c.st, c.S, (long long)r * r));   // also clears S
    MAPL_RETURN_IF(tc_st_split(G, d, r, batch, 0, 0.f, nullptr, c.Ptr2, c.st));
    MAPL_RETURN_IF(tc_st_gemm3(c.Ptr, c.Ptr2, r, r, d, batch, c.S, nullptr, 0.f, (d / 64 + 3) / 4, c.st));
    MAPL_RETURN_IF(tc_st_split(c.S, r, r, batch, 3, 0.f, c.Pm, nullptr, c.st));
    return tc_st_gemm3(c.Prow, c.Pm, d, r, r, batch, out, G, 1.f, 1, c.st);
  }
  MAPL_RETURN_IF(gram(U, G, c.S, d, r, batch, c.st));
  { KernelScope ks(KID_ST_STEP_MATRIX, c.st); k_neg_sym<<<dim3((r * r + 255) / 256, batch), 256, 0, c.st>>>(c.S, c.M, r); }
  MAPL_CUDA_CHECK(cudaGetLastError());
  return right_mul(U, c.M, out, G, 1.f, d, r, batch, c.st);
}

// `iters` cubic Newton-Schulz iterations X <- X (3I - X^T X)/2 from `cur` (overwritten) with scratch `nxt`; the last
// iterate is written to `final_out` (which may be neither cur nor nxt)
int ctx_ns(const StCtx& c, float* cur, float* nxt, float* final_out, int iters) {
  const int d = c.d, r = c.r, batch = c.batch;
  for (int it = 0; it < iters; ++it) {
    float* out = (it == iters - 1) ? final_out : nxt;
    if (c.tc) {
      MAPL_RETURN_IF(tc_st_split(cur, d, r, batch, 0, 0.f, c.Prow, c.Ptr, c.st, c.S, (long long)r * r));
      MAPL_RETURN_IF(tc_st_gemm3(c.Ptr, c.Ptr, r, r, d, batch, c.S, nullptr, 0.f, (d / 64 + 3) / 4, c.st));
      MAPL_RETURN_IF(tc_st_split(c.S, r, r, batch, 1, 0.f, c.Pm, nullptr, c.st));
      MAPL_RETURN_IF(tc_st_gemm3(c.Prow, c.Pm, d, r, r, batch, out, nullptr, 0.f, 1, c.st));
    } else {
      MAPL_RETURN_IF(gram(cur, cur, c.S, d, r, batch, c.st, true));
      { KernelScope ks(KID_ST_NS_POLY, c.st); k_ns_poly<<<dim3((r * r + 255) / 256, batch), 256, 0, c.st>>>(c.S, c.M, r); }
      MAPL_CUDA_CHECK(cudaGetLastError());
      MAPL_RETURN_IF(right_mul(cur, c.M, out, nullptr, 0.f, d, r, batch, c.st));
    }
    nxt = cur; cur = out;
  }
  return MAPL_OK;
}

}  // namespace

int st_gemm_nn(const float* A, const float* B, float* C, int M, int N, int K, cudaStream_t st, float alpha, const float* E,
               float beta) {
  if (M <= 0 || N <= 0 || K <= 0) return MAPL_OK;
  if (N % 4 || K % 4) return MAPL_ERR_UNSUPPORTED;
  const int tiles = ((M + TM - 1) / TM) * ((N + TN - 1) / TN);
  KernelScope ks(KID_ST_GEMM, st);
  k_st_gemm<false><<<dim3(tiles, 1, 1), 256, 0, st>>>(A, B, C, E, alpha, beta, M, N, K, K, 0, 0, 0, 0, K, N, N);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

int st_gemm_tn(const float* X, const float* Y, float* C, int M, int N, int K, cudaStream_t st, float alpha) {
  if (M <= 0 || N <= 0 || K <= 0) return MAPL_OK;
  if (M % 4 || N % 4) return MAPL_ERR_UNSUPPORTED;
  const int tiles = ((M + TM - 1) / TM) * ((N + TN - 1) / TN);
  int splits = (2 * 148 + tiles - 1) / tiles;
  int kper = ((K + splits - 1) / splits + TK - 1) / TK * TK;
  if (kper < 4 * TK) kper = 4 * TK;
  splits = (K + kper - 1) / kper;
  KernelScope ks(KID_ST_GEMM, st);
  k_st_gemm<true><<<dim3(tiles, splits, 1), 256, 0, st>>>(X, Y, C, nullptr, alpha, 0.f, M, N, K, kper, 0, 0, 0, 0, M, N, N);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

}  // namespace mapl

using namespace mapl;

extern "C" {

size_t mapl_stiefel_workspace_bytes(int32_t d, int32_t r, int32_t batch) {
  if (d < 8 || r < 8 || r > d || d % 8 || r % 8 || batch < 1 || r > 1024) return 0;
  return st_carve(d, r, batch).total;
}

int mapl_stiefel_step(int32_t d, int32_t r, int32_t batch, float* U, const float* G, float lr,
                      int32_t retraction, int32_t ns_iters, float* info_out, void* workspace,
                      size_t workspace_bytes, void* cuda_stream) {
  if (d < 8 || r < 8 || r > d || d % 8 || r % 8 || batch < 1) return MAPL_ERR_INVALID_ARG;
  if (r > 1024) return MAPL_ERR_UNSUPPORTED;
  if (!U || !G) return MAPL_ERR_INVALID_ARG;
  if (retraction != MAPL_RETRACT_QR && retraction != MAPL_RETRACT_NS) return MAPL_ERR_INVALID_ARG;
  if (retraction == MAPL_RETRACT_NS && (ns_iters < 1 || ns_iters > 16)) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(U) || !aligned16(G) || !aligned16(workspace) || (info_out && !aligned16(info_out)))
    return MAPL_ERR_ALIGNMENT;
  const StWs w = st_carve(d, r, batch);
  if (!workspace || workspace_bytes < w.total) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = reinterpret_cast<char*>(workspace);
  float* S = reinterpret_cast<float*>(ws + w.S);
  float* M = reinterpret_cast<float*>(ws + w.M);
  float* Rinv = reinterpret_cast<float*>(ws + w.Rinv);
  float* Rinv2 = reinterpret_cast<float*>(ws + w.Rinv2);
  float* X0 = reinterpret_cast<float*>(ws + w.X0);
  float* X1 = reinterpret_cast<float*>(ws + w.X1);
  const dim3 egrid((r * r + 255) / 256, batch);

  // ---- tensor-core path (d and r multiples of 128, r >= 256): every [d,r]-sized GEMM of the step as six bf16-plane
  // MMAs (tc_stiefel.cu); MAPL_ST_TC=0 forces the FFMA kernels (debugging aid)
  static const bool tc_enabled = !(getenv("MAPL_ST_TC") && getenv("MAPL_ST_TC")[0] == '0');
  if (tc_st_ok(d, r) && tc_enabled) {
    __nv_bfloat16* Prow = reinterpret_cast<__nv_bfloat16*>(ws + w.Prow);   // [b][3][d][r]
    __nv_bfloat16* Ptr = reinterpret_cast<__nv_bfloat16*>(ws + w.Ptr);     // [b][3][r][d]
    __nv_bfloat16* Ptr2 = reinterpret_cast<__nv_bfloat16*>(ws + w.Ptr2);   // [b][3][r][d]
    __nv_bfloat16* Pm = reinterpret_cast<__nv_bfloat16*>(ws + w.Pm);       // [b][3][r][r]
    // Gram products: at most 4 k-blocks of 64 per CTA, one per TMEM accumulator.  A longer chain of MMAs into one
    // accumulator shows the tensor core's truncating accumulate on diag(X^T X): d = 384 with d / 256 = 1 split ran 6
    // k-blocks in one CTA and left ||U^T U - I||_F = 1.3e-5 (3.4e-6 with two splits of 3).
    const int ksplit = (d / 64 + 3) / 4;
    // S = U^T G ;  M1 = I + lr sym(S) ;  Y = U M1 - lr G  -> X0   (the split of U also clears S: no memset node, which
    // would break the chain of programmatic dependent launches)
    MAPL_RETURN_IF(tc_st_split(U, d, r, batch, 0, 0.f, Prow, Ptr, st, S, (long long)r * r));
    MAPL_RETURN_IF(tc_st_split(G, d, r, batch, 0, 0.f, nullptr, Ptr2, st));
    MAPL_RETURN_IF(tc_st_gemm3(Ptr, Ptr2, r, r, d, batch, S, nullptr, 0.f, ksplit, st));
    MAPL_RETURN_IF(tc_st_split(S, r, r, batch, 2, lr, Pm, nullptr, st));     // M1 is symmetric: its planes are B^T too
    MAPL_RETURN_IF(tc_st_gemm3(Prow, Pm, d, r, r, batch, X0, G, -lr, 1, st));
    if (info_out) {
      KernelScope ks(KID_ST_FRO_NORM, st);
      k_fro_norm<<<batch, 1024, 0, st>>>(U, X0, lr != 0.f ? 1.f / lr : 0.f, (long long)d * r, 0, info_out, 0);
      MAPL_CUDA_CHECK(cudaGetLastError());
    }
    if (retraction == MAPL_RETRACT_QR) {     // CholeskyQR2 (see the FFMA path below); Gram and X R^-1 on the tensor cores
      const float* src = X0;
      for (int pass = 0; pass < 2; ++pass) {
        MAPL_RETURN_IF(tc_st_split(src, d, r, batch, 0, 0.f, Prow, Ptr, st, S, (long long)r * r));   // also clears S
        MAPL_RETURN_IF(tc_st_gemm3(Ptr, Ptr, r, r, d, batch, S, nullptr, 0.f, ksplit, st));           // X^T X
        MAPL_RETURN_IF(chol_inverse_blocked(S, Rinv, M, Rinv2, r, batch, st));
        MAPL_RETURN_IF(tc_st_split(Rinv, r, r, batch, 0, 0.f, nullptr, Pm, st));                      // planes of (R^-1)^T
        float* out = pass == 0 ? X1 : U;
        MAPL_RETURN_IF(tc_st_gemm3(Prow, Pm, d, r, r, batch, out, nullptr, 0.f, 1, st));
        src = out;
      }
    }
    float* cur = X0;
    float* nxt = X1;
    for (int it = 0; it < (retraction == MAPL_RETRACT_NS ? ns_iters : 0); ++it) {
      MAPL_RETURN_IF(tc_st_split(cur, d, r, batch, 0, 0.f, Prow, Ptr, st, S, (long long)r * r));   // also clears S
      MAPL_RETURN_IF(tc_st_gemm3(Ptr, Ptr, r, r, d, batch, S, nullptr, 0.f, ksplit, st));   // X^T X
      MAPL_RETURN_IF(tc_st_split(S, r, r, batch, 1, 0.f, Pm, nullptr, st));                 // (3I - X^T X)/2, symmetric
      float* out = (it == ns_iters - 1) ? U : nxt;
      MAPL_RETURN_IF(tc_st_gemm3(Prow, Pm, d, r, r, batch, out, nullptr, 0.f, 1, st));
      nxt = cur; cur = out;
    }
    if (info_out) {
      MAPL_RETURN_IF(gram(U, U, S, d, r, batch, st));
      KernelScope ks(KID_ST_FRO_NORM, st);
      k_fro_norm<<<batch, 1024, 0, st>>>(S, nullptr, 1.f, (long long)r * r, r, info_out, 1);
      MAPL_CUDA_CHECK(cudaGetLastError());
    }
    return MAPL_OK;
  }

  // tangent projection + step:  Y = U (I + lr sym(U^T G)) - lr G   -> X0
  MAPL_RETURN_IF(gram(U, G, S, d, r, batch, st));
  { KernelScope ks(KID_ST_STEP_MATRIX, st); k_step_matrix<<<egrid, 256, 0, st>>>(S, M, r, lr); }
  MAPL_CUDA_CHECK(cudaGetLastError());
  MAPL_RETURN_IF(right_mul(U, M, X0, G, -lr, d, r, batch, st));
  if (info_out) {   // ||xi||_F = ||U - Y||_F / lr
    KernelScope ks(KID_ST_FRO_NORM, st);
    k_fro_norm<<<batch, 1024, 0, st>>>(U, X0, lr != 0.f ? 1.f / lr : 0.f, (long long)d * r, 0, info_out, 0);
    MAPL_CUDA_CHECK(cudaGetLastError());
  }

  if (retraction == MAPL_RETRACT_NS) {
    float* cur = X0;
    float* nxt = X1;
    for (int it = 0; it < ns_iters; ++it) {
      MAPL_RETURN_IF(gram(cur, cur, S, d, r, batch, st, true));
      { KernelScope ks(KID_ST_NS_POLY, st); k_ns_poly<<<egrid, 256, 0, st>>>(S, M, r); }
      MAPL_CUDA_CHECK(cudaGetLastError());
      float* out = (it == ns_iters - 1) ? U : nxt;
      MAPL_RETURN_IF(right_mul(cur, M, out, nullptr, 0.f, d, r, batch, st));
      nxt = cur; cur = out;
    }
  } else {
    // CholeskyQR2: Y = Q1 R1, Q1 = Q R2  =>  Y = Q (R2 R1), upper triangular with positive diagonal
    const float* src = X0;
    for (int pass = 0; pass < 2; ++pass) {
      MAPL_RETURN_IF(gram(src, src, S, d, r, batch, st, true));   // the factorisation reads the upper triangle only
      MAPL_RETURN_IF(chol_inverse_blocked(S, Rinv, M, Rinv2, r, batch, st));
      float* Xinv = Rinv;
      float* out = pass == 0 ? X1 : U;
      MAPL_RETURN_IF(right_mul(src, Xinv, out, nullptr, 0.f, d, r, batch, st));
      src = out;
    }
  }
  if (info_out) {   // ||U^T U - I||_F
    MAPL_RETURN_IF(gram(U, U, S, d, r, batch, st));
    KernelScope ks(KID_ST_FRO_NORM, st);
    k_fro_norm<<<batch, 1024, 0, st>>>(S, nullptr, 1.f, (long long)r * r, r, info_out, 1);
    MAPL_CUDA_CHECK(cudaGetLastError());
  }
  return MAPL_OK;
}

size_t mapl_spel_workspace_bytes(int32_t d, int32_t r, int32_t batch) { return mapl_stiefel_workspace_bytes(d, r, batch); }

int mapl_spel_step(int32_t d, int32_t r, int32_t batch, float* U, const float* G, float* Mom, float lr, float beta,
                   int32_t lmo_iters, int32_t retr_iters, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (d < 8 || r < 8 || r > d || d % 8 || r % 8 || batch < 1) return MAPL_ERR_INVALID_ARG;
  if (r > 1024) return MAPL_ERR_UNSUPPORTED;
  if (!U || !G || !Mom) return MAPL_ERR_INVALID_ARG;
  if (lmo_iters < 1 || lmo_iters > 16 || retr_iters < 1 || retr_iters > 16) return MAPL_ERR_INVALID_ARG;
  if (!(beta >= 0.f && beta <= 1.f)) return MAPL_ERR_INVALID_ARG;
  if (!aligned16(U) || !aligned16(G) || !aligned16(Mom) || !aligned16(workspace)) return MAPL_ERR_ALIGNMENT;
  const StWs w = st_carve(d, r, batch);
  if (!workspace || workspace_bytes < w.total) return MAPL_ERR_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = reinterpret_cast<char*>(workspace);
  float* X0 = reinterpret_cast<float*>(ws + w.X0);
  float* X1 = reinterpret_cast<float*>(ws + w.X1);
  float* X2 = reinterpret_cast<float*>(ws + w.X2);
  float* norm2 = reinterpret_cast<float*>(ws + w.norm2);
  static const bool tc_enabled = !(getenv("MAPL_ST_TC") && getenv("MAPL_ST_TC")[0] == '0');
  StCtx c;
  c.d = d; c.r = r; c.batch = batch; c.st = st; c.tc = tc_st_ok(d, r) && tc_enabled;
  c.S = reinterpret_cast<float*>(ws + w.S); c.M = reinterpret_cast<float*>(ws + w.M);
  c.Prow = reinterpret_cast<__nv_bfloat16*>(ws + w.Prow); c.Ptr = reinterpret_cast<__nv_bfloat16*>(ws + w.Ptr);
  c.Ptr2 = reinterpret_cast<__nv_bfloat16*>(ws + w.Ptr2); c.Pm = reinterpret_cast<__nv_bfloat16*>(ws + w.Pm);
  const long long n = (long long)d * r;
  const dim3 eg(148, batch);

  MAPL_RETURN_IF(ctx_tangent(c, U, G, X0));                                                   // Eq. 4: xi -> X0
  { KernelScope ks(KID_MEMSET, st); MAPL_CUDA_CHECK(cudaMemsetAsync(norm2, 0, (size_t)batch * 4, st)); }
  { KernelScope ks(KID_ST_STEP_MATRIX, st); k_momentum<<<eg, 256, 0, st>>>(Mom, X0, beta, n, norm2); }     // Eq. 5
  MAPL_CUDA_CHECK(cudaGetLastError());
  { KernelScope ks(KID_ST_STEP_MATRIX, st); k_axpby_scaled<<<eg, 256, 0, st>>>(X1, nullptr, 0.f, Mom, 1.f, norm2, n); }   // m / ||m||_F
  MAPL_CUDA_CHECK(cudaGetLastError());
  MAPL_RETURN_IF(ctx_ns(c, X1, X0, X2, lmo_iters));                                           // Eq. 6: d_t -> X2
  { KernelScope ks(KID_ST_STEP_MATRIX, st); k_axpby_scaled<<<eg, 256, 0, st>>>(X0, U, 1.f, X2, -lr, nullptr, n); }        // U - lr d_t
  MAPL_CUDA_CHECK(cudaGetLastError());
  return ctx_ns(c, X0, X1, U, retr_iters);                                                    // Eq. 7
}

}  // extern "C"
