// profile.cu -- see profile.cuh.
#include <vector>

#include "common.cuh"
#include "profile.cuh"

namespace mapl {
namespace {

const char* kNames[KID_COUNT] = {
    "k_simt_gemm", "k_half_sqnorm", "k_simt_encode_rvq", "k_dequant", "k_scatter_add_rows",
    "k_step_matrix", "k_ns_poly", "k_fro_norm", "k_chol_upper", "k_tri_inverse_upper", "memset",
    "k_tc_pack", "k_tc_encode", "k_tc_decode", "k_tc_bwd_gz", "k_tc_bwd_du", "k_tc_encode_rvq",
    "k_tc_scatter", "k_st_gemm", "k_st_split", "k_tc_gemm3", "k_mcvq", "k_stream_diag"};

struct Pair { cudaEvent_t a, b; int kid; };
bool g_timing = false;
long long g_count[KID_COUNT] = {0};
double g_ms[KID_COUNT] = {0};
long long g_timed[KID_COUNT] = {0};
std::vector<Pair> g_pending;
std::vector<cudaEvent_t> g_pool;

cudaEvent_t get_event() {
  if (!g_pool.empty()) { cudaEvent_t e = g_pool.back(); g_pool.pop_back(); return e; }
  cudaEvent_t e;
  cudaEventCreate(&e);
  return e;
}

void drain() {
  for (Pair& p : g_pending) {
    float ms = 0.f;
    if (cudaEventSynchronize(p.b) == cudaSuccess && cudaEventElapsedTime(&ms, p.a, p.b) == cudaSuccess) {
      g_ms[p.kid] += ms;
      g_timed[p.kid] += 1;
    }
    g_pool.push_back(p.a);
    g_pool.push_back(p.b);
  }
  g_pending.clear();
}

}  // namespace

void prof_begin(int kid, cudaStream_t st) {
  g_count[kid] += 1;
  if (!g_timing) return;
  Pair p{get_event(), get_event(), kid};
  cudaEventRecord(p.a, st);
  g_pending.push_back(p);
}

void prof_end(int kid, cudaStream_t st) {
  if (!g_timing) return;
  (void)kid;
  cudaEventRecord(g_pending.back().b, st);
}

}  // namespace mapl

using namespace mapl;

extern "C" {

int mapl_profile_kernel_count(void) { return KID_COUNT; }

const char* mapl_profile_kernel_name(int kid) { return (kid >= 0 && kid < KID_COUNT) ? kNames[kid] : ""; }

void mapl_profile_enable(int timing_on) {
  if (!timing_on && g_timing) drain();
  g_timing = timing_on != 0;
}

void mapl_profile_reset(void) {
  drain();
  for (int i = 0; i < KID_COUNT; ++i) { g_count[i] = 0; g_ms[i] = 0; g_timed[i] = 0; }
}

int mapl_profile_read(int kid, long long* launches, long long* timed_launches, double* total_ms) {
  if (kid < 0 || kid >= KID_COUNT) return MAPL_ERR_INVALID_ARG;
  drain();
  if (launches) *launches = g_count[kid];
  if (timed_launches) *timed_launches = g_timed[kid];
  if (total_ms) *total_ms = g_ms[kid];
  return MAPL_OK;
}

}  // extern "C"
