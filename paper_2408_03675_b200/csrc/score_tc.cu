// score_tc.cu -- tensor-core scoring path (placeholder until the tcgen05 kernels land).
#include "nacl_internal.cuh"

namespace nacl {
bool score_tc_supported(const Shape&) { return false; }
int score_tc_launch_count(const Shape&) { return 0; }
cudaError_t launch_score_tc(const Shape&, const void*, const void*, const SplitPlan&, const Workspace&, float*, float*,
                            cudaStream_t) {
  return cudaErrorNotSupported;
}
}  // namespace nacl
