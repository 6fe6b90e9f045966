// nb_small_launch.h -- what nbody_b200.cu needs of the small-call kernel's translation unit (nb_small_launch.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

namespace nb {
struct SmallArgs;
struct SmallPlan;
// One launch of nb_small_kernel under plan p.  mode = SMALL_EXACT (every pair masked), SMALL_FLAG (pairs marked while
// staged, only those masked; needs eps2 >= 2^-40; falls back to SMALL_EXACT for LJ > 1) or SMALL_NONE (no mask, no
// potential: valid when pot == nullptr and eps2 >= 2^-40) -- nb_small.cuh.
cudaError_t small_launch(const SmallPlan& p, SmallArgs a, int mode, cudaStream_t stream);
}  // namespace nb
