// placeholder until the tcgen05 forward lands
#include "common.cuh"
namespace strata {
bool tc_fwd_supported(const Problem&) { return false; }
cudaError_t launch_fwd_tc(const Problem&, const void*, const void*, const void*, void*, float*, cudaStream_t, int*) {
  return cudaErrorNotSupported;
}
}  // namespace strata
