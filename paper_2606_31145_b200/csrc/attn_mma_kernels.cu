// bf16 tensor-core (mma.sync) kernels for stage 1 / stage 2 -- placeholder until implemented.
#include "sekv_internal.cuh"

namespace sekv {
bool have_mma_kernels() { return false; }
cudaError_t launch_stage1_mma(sekv_handle*, int, const void*, cudaStream_t) { return cudaErrorNotSupported; }
cudaError_t launch_stage2_mma(sekv_handle*, int, const void*, const int32_t*, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace sekv
