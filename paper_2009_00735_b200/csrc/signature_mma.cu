// signature_mma.cu -- windowed-DFT signature kernel on the tcgen05 tensor cores (narrow windows).
// Placeholder until the kernel lands: reports "not supported" so plans use the FFT kernel.
#include "common.cuh"

namespace apx {
bool mma_path_supported(const Plan *) { return false; }
cudaError_t mma_path_prepare(Plan *) { return cudaSuccess; }
cudaError_t launch_signature_mma(Plan *, const float *, int64_t, float *, uint32_t *, cudaStream_t)
{
    return cudaErrorNotSupported;
}
}  // namespace apx
