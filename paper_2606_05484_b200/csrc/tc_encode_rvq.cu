// tc_encode_rvq.cu -- placeholder until the fused projection + RVQ tcgen05 kernel lands.
#include "tc_codec.cuh"
namespace mapl {
int tc_encode_rvq(const mapl_boundary_desc&, const void*, const float*, const TcPack&, void*, int32_t*, cudaStream_t) {
  return MAPL_ERR_UNSUPPORTED;
}
}  // namespace mapl
