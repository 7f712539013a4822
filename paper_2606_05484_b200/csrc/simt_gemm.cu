// simt_gemm.cu -- generic fp32-FFMA tiled GEMM used by the general path of libmapl (any shape,
// fp32 or bf16 operands, optional row/k gather, split-K with atomics, batched).  It is the path
// that meets the 1e-5 fp32 tolerance (tcgen05 has no fp32 MMA kind) and the fallback for shapes
// the tensor-core kernels do not take.
#include "common.cuh"
#include "profile.cuh"

namespace mapl {

thread_local int g_last_cuda_error = 0;

namespace {

constexpr int BM = 64, BN = 64, BK = 16, NT = 256, PAD = 4;

struct DevMat {
  const void* p; int bf16; long long so, sk; const int32_t* gather; int gmode;
};
struct DevGemm {
  int M, N, npairs;
  DevMat A[2], B[2];
  int K[2];
  void* C; int c_bf16; long long ldc, sbc;
  int splits, atomic;
  float alpha; const float* E; long long lde, sbe; float beta; const int32_t* e_gather;
  long long sbA[2], sbB[2];
};

// load a [BK x 64] tile of operand `m` (outer offset o0, k offset k0) into s[k][i]
__device__ __forceinline__ void load_tile(float (*s)[BM + PAD], const DevMat& m, long long batch_off,
                                          int o0, int omax, int k0, int kmax) {
  const int t = threadIdx.x;
  if (m.sk == 1) {  // k contiguous: consecutive threads walk k
#pragma unroll
    for (int it = 0; it < (BM * BK) / NT; ++it) {
      int idx = t + it * NT;
      int k = idx % BK, i = idx / BK;
      int go = o0 + i, gk = k0 + k;
      float v = 0.f;
      if (go < omax && gk < kmax) {
        long long oi = (m.gmode == 1) ? (long long)m.gather[go] : (long long)go;
        long long ki = (m.gmode == 2) ? (long long)m.gather[gk] : (long long)gk;
        v = ld_as_f32(m.p, batch_off + oi * m.so + ki * m.sk, m.bf16);
      }
      s[k][i] = v;
    }
  } else {          // outer index contiguous (or general strides): consecutive threads walk i
#pragma unroll
    for (int it = 0; it < (BM * BK) / NT; ++it) {
      int idx = t + it * NT;
      int i = idx % BM, k = idx / BM;
      int go = o0 + i, gk = k0 + k;
      float v = 0.f;
      if (go < omax && gk < kmax) {
        long long oi = (m.gmode == 1) ? (long long)m.gather[go] : (long long)go;
        long long ki = (m.gmode == 2) ? (long long)m.gather[gk] : (long long)gk;
        v = ld_as_f32(m.p, batch_off + oi * m.so + ki * m.sk, m.bf16);
      }
      s[k][i] = v;
    }
  }
}

__global__ void __launch_bounds__(NT) k_simt_gemm(const DevGemm g) {
  __shared__ __align__(16) float As[BK][BM + PAD];
  __shared__ __align__(16) float Bs[BK][BN + PAD];
  const int tiles_n = (g.N + BN - 1) / BN;
  const int tm = blockIdx.x / tiles_n, tn = blockIdx.x % tiles_n;
  const int split = blockIdx.y, b = blockIdx.z;
  const int m0 = tm * BM, n0 = tn * BN;
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int p = 0; p < g.npairs; ++p) {
    const int K = g.K[p];
    // split the k range in BK-aligned chunks
    const int nkb = (K + BK - 1) / BK;
    const int per = (nkb + g.splits - 1) / g.splits;
    const int kb0 = split * per, kb1 = min(nkb, kb0 + per);
    const long long offA = (long long)b * g.sbA[p], offB = (long long)b * g.sbB[p];
    for (int kb = kb0; kb < kb1; ++kb) {
      load_tile(As, g.A[p], offA, m0, g.M, kb * BK, K);
      load_tile(Bs, g.B[p], offB, n0, g.N, kb * BK, K);
      __syncthreads();
#pragma unroll
      for (int k = 0; k < BK; ++k) {
        const float4 a = *reinterpret_cast<const float4*>(&As[k][ty * 4]);
        const float4 bb = *reinterpret_cast<const float4*>(&Bs[k][tx * 4]);
        const float av[4] = {a.x, a.y, a.z, a.w};
        const float bv[4] = {bb.x, bb.y, bb.z, bb.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
      }
      __syncthreads();
    }
  }
  const long long offC = (long long)b * g.sbc, offE = (long long)b * g.sbe;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i;
    if (m >= g.M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= g.N) continue;
      float v = g.alpha * acc[i][j];
      const long long ci = offC + (long long)m * g.ldc + n;
      if (g.atomic) {
        atomicAdd(reinterpret_cast<float*>(g.C) + ci, v);
      } else {
        if (g.E) v += g.beta * g.E[offE + (long long)(g.e_gather ? g.e_gather[m] : m) * g.lde + n];
        st_from_f32(g.C, ci, g.c_bf16, v);
      }
    }
  }
}

}  // namespace

int simt_gemm(const GemmArgs& a, cudaStream_t stream) {
  if (a.M <= 0 || a.N <= 0 || a.batch <= 0) return MAPL_OK;
  if (a.splits > 1 && !a.atomic) return MAPL_ERR_INVALID_ARG;
  if (a.atomic && (a.c_bf16 || a.E)) return MAPL_ERR_INVALID_ARG;
  DevGemm g;
  g.M = a.M; g.N = a.N; g.npairs = a.npairs;
  for (int p = 0; p < 2; ++p) {
    g.A[p] = DevMat{a.A[p].p, a.A[p].bf16, a.A[p].so, a.A[p].sk, a.A[p].gather, a.A[p].gmode};
    g.B[p] = DevMat{a.B[p].p, a.B[p].bf16, a.B[p].so, a.B[p].sk, a.B[p].gather, a.B[p].gmode};
    g.K[p] = a.K[p];
    g.sbA[p] = a.A[p].sb; g.sbB[p] = a.B[p].sb;
  }
  g.C = a.C; g.c_bf16 = a.c_bf16; g.ldc = a.ldc; g.sbc = a.sbc;
  g.splits = a.splits < 1 ? 1 : a.splits; g.atomic = a.atomic;
  g.alpha = a.alpha; g.E = a.E; g.lde = a.lde; g.sbe = a.sbe; g.beta = a.beta; g.e_gather = a.e_gather;
  const int tiles = ((a.M + BM - 1) / BM) * ((a.N + BN - 1) / BN);
  dim3 grid(tiles, g.splits, a.batch);
  { KernelScope ks(KID_SIMT_GEMM, stream); k_simt_gemm<<<grid, NT, 0, stream>>>(g); }
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

}  // namespace mapl
