#include "tc_codec.cuh"
namespace mapl {
int tc_decode(const mapl_boundary_desc&, const void*, const int32_t*, const float*, const float*,
              const int32_t*, const float*, const float*, void*, char*, cudaStream_t) {
  return MAPL_ERR_UNSUPPORTED;
}
}  // namespace mapl
