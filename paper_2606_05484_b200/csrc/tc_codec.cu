// tc_codec.cu -- envelope checks, parameter packing and workspace layout shared by the tcgen05 codec
// kernels (tc_encode.cu, tc_decode.cu, tc_backward.cu).
#include "tc_codec.cuh"

#include "profile.cuh"

namespace mapl {

bool tc_shape_ok(const mapl_boundary_desc& d) {
  if (d.act_dtype != MAPL_BF16) return false;
  if (d.d % 128 != 0 || d.d < 128) return false;
  if (d.r != 64 && d.r != 128 && d.r != 256) return false;
  if (d.anchor_rank != 0 && d.anchor_rank != 64 && d.anchor_rank != 128) return false;
  if (d.n_tokens < 1) return false;
  return true;
}

size_t tc_workspace_bytes(const mapl_boundary_desc& d) {
  if (!tc_shape_ok(d)) return 0;
  const size_t pack = align_up((size_t)(d.r + d.anchor_rank) * d.d * 2, 256);
  // + bf16 zhat [N, r] materialised from RVQ codes for the dU operand of backward
  return 2 * pack + (d.rvq_levels > 0 ? align_up((size_t)d.n_tokens * d.r * 2, 256) : 0);
}

TcPacks tc_packs(const mapl_boundary_desc& d, char* tc_ws) {
  const size_t pack = align_up((size_t)(d.r + d.anchor_rank) * d.d * 2, 256);
  TcPacks p;
  p.WB = reinterpret_cast<__nv_bfloat16*>(tc_ws);
  p.Wd = reinterpret_cast<__nv_bfloat16*>(tc_ws + pack);
  p.kc = d.r + d.anchor_rank;
  return p;
}

namespace {

struct PackJob {
  const float* src; int rows, cols;        // src is [rows, cols] fp32 row-major
  __nv_bfloat16* dst; long long pitch;     // dst element (i,j) -> dst[i*pitch + j] (after optional transpose)
  int transpose;
};
struct PackArgs { PackJob job[4]; int njobs; };

// 32x32 tiles; blockIdx.y = job
__global__ void __launch_bounds__(256) k_tc_pack(const PackArgs a) {
  __shared__ float tile[32][33];
  const PackJob j = a.job[blockIdx.y];
  const int tiles_c = (j.cols + 31) / 32, tiles_r = (j.rows + 31) / 32;
  for (int t = blockIdx.x; t < tiles_c * tiles_r; t += gridDim.x) {
    const int r0 = (t / tiles_c) * 32, c0 = (t % tiles_c) * 32;
    const int tx = threadIdx.x % 32, ty = threadIdx.x / 32;
    for (int i = ty; i < 32; i += 8) {
      const int r = r0 + i, c = c0 + tx;
      tile[i][tx] = (r < j.rows && c < j.cols) ? j.src[(long long)r * j.cols + c] : 0.f;
    }
    __syncthreads();
    if (j.transpose) {
      for (int i = ty; i < 32; i += 8) {
        const int c = c0 + i, r = r0 + tx;           // dst row = src col
        if (c < j.cols && r < j.rows) j.dst[(long long)c * j.pitch + r] = __float2bfloat16_rn(tile[tx][i]);
      }
    } else {
      for (int i = ty; i < 32; i += 8) {
        const int r = r0 + i, c = c0 + tx;
        if (r < j.rows && c < j.cols) j.dst[(long long)r * j.pitch + c] = __float2bfloat16_rn(tile[i][tx]);
      }
    }
    __syncthreads();
  }
}

}  // namespace

int tc_pack_params(const mapl_boundary_desc& d, const float* U, const float* B, const TcPacks& p, int which,
                   cudaStream_t st) {
  PackArgs a;
  a.njobs = 0;
  const int ra = d.anchor_rank;
  if (which & 1) a.job[a.njobs++] = PackJob{U, d.d, d.r, p.WB, d.d, 1};                               // WB[j][i] = U[i][j]
  if ((which & 2) && ra && B) a.job[a.njobs++] = PackJob{B, ra, d.d, p.WB + (long long)d.r * d.d, d.d, 0};
  if (which & 4) a.job[a.njobs++] = PackJob{U, d.d, d.r, p.Wd, p.kc, 0};                              // Wd[i][j] = U[i][j]
  if ((which & 8) && ra && B) a.job[a.njobs++] = PackJob{B, ra, d.d, p.Wd + d.r, p.kc, 1};            // Wd[i][r+q] = B[q][i]
  if (a.njobs == 0) return MAPL_OK;
  KernelScope ks(KID_TC_PACK, st);
  k_tc_pack<<<dim3(128, a.njobs), 256, 0, st>>>(a);
  MAPL_CUDA_CHECK(cudaGetLastError());
  return MAPL_OK;
}

}  // namespace mapl
