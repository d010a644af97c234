// step_tiled.cu -- tiled fused kick+drift kernel (placeholder until the z-marching kernel lands).
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {
bool step_tiled_supports(int) { return false; }
cudaError_t launch_step_tiled(const Lattice &, const StepCoef &, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace u1u1
