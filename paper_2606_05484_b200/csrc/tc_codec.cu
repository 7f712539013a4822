// tc_codec.cu -- dispatch of the tcgen05 codec kernels (placeholder until the kernels land).
#include "tc_codec.cuh"

namespace mapl {

size_t tc_workspace_bytes(const mapl_boundary_desc&) { return 0; }

int tc_encode(const mapl_boundary_desc&, const void*, const float*, const float*, void*, int32_t*, char*,
              cudaStream_t) { return MAPL_ERR_UNSUPPORTED; }

int tc_decode(const mapl_boundary_desc&, const void*, const int32_t*, const float*, const float*,
              const int32_t*, const float*, const float*, void*, char*, cudaStream_t) {
  return MAPL_ERR_UNSUPPORTED;
}

int tc_backward(const mapl_boundary_desc&, const void*, const void*, const void*, const int32_t*, const float*,
                const float*, const int32_t*, const float*, const float*, void*, float*, float*, float*, void*,
                char*, float*, cudaStream_t) {
  return MAPL_ERR_UNSUPPORTED;
}

}  // namespace mapl
