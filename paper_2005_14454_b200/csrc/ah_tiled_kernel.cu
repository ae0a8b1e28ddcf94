// ah_tiled_kernel.cu — placeholder until the z-marching kernel lands (next commit).
#include "ah_kernels.h"

namespace ah {
bool tiled_supported(int, int, int) { return false; }
cudaError_t tiled_setup() { return cudaSuccess; }
cudaError_t launch_tiled_step(const ConstFields<float> &, const Fields<float> &, const StepCoef<float> &,
                              int, int, int, cudaStream_t)
{
    return cudaErrorNotSupported;
}
}  // namespace ah
