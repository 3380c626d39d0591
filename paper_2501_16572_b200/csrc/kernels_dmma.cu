// Fast variant (EXX_VARIANT_FUSED_DMMA) -- placeholder until the tensor-core kernels land.
#include "exx_internal.h"

namespace exx {
cudaError_t fast_init(exx_plan*) { return cudaSuccess; }
void fast_destroy(exx_plan*) {}
cudaError_t fast_solve_batch(exx_plan*, double*, double*, int, const FastArgs*, cudaStream_t, long long*) {
  return cudaErrorNotSupported;
}
}  // namespace exx
