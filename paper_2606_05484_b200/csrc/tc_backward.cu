#include "tc_codec.cuh"
namespace mapl {
int tc_backward(const mapl_boundary_desc&, const void*, const void*, const void*, const int32_t*, const float*,
                const float*, const int32_t*, const float*, const float*, void*, float*, float*, float*, void*,
                char*, float*, cudaStream_t) {
  return MAPL_ERR_UNSUPPORTED;
}
}  // namespace mapl
