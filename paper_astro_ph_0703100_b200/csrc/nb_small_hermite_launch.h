// nb_small_hermite_launch.h -- what nbody_b200.cu needs of the small-i-set force + jerk kernel's translation unit.
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

namespace nb {
struct SmallHermiteArgs;
struct SmallPlan;
// One launch of nb_small_hermite_kernel under plan p (KI = 1; the shapes of small_jerk_shape_ok, nb_plan.h); every pair masked.
cudaError_t small_hermite_launch(const SmallPlan& p, const SmallHermiteArgs& a, cudaStream_t stream);
}  // namespace nb
