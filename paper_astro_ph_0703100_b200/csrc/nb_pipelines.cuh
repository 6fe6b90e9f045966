// nb_pipelines.cuh -- the paper's two pipeline descriptions, statement by statement, and a Lennard-Jones pipeline, as
// pipelines of the generalised kernel (include/nb_pipeline.cuh).  The only addition to the listings is the coincident-pair rule
// (reading R1): a pair whose three position differences are exactly zero adds nothing.
#pragma once
#include "../../include/nb_pipeline.cuh"

namespace nb {

// 1/sqrt as one MUFU.RSQ (the listings' "1/sqrt(r2)"; same instruction as the specialised kernels)
__device__ __forceinline__ float pipeline_rsqrt(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Fig. A.1 / A.3: IDIM 4 = (x, y, z, eps2), JDIM 4 = (x, y, z, m), FDIM 3 = (ax, ay, az)
struct PipelineForceA3 {
    static constexpr int IDIM = 4, JDIM = 4, FDIM = 3;
    static __device__ __forceinline__ void pair(const float* INPUT_I, const float* INPUT_J, float* OUTPUT) {
        const float xi = INPUT_I[0], yi = INPUT_I[1], zi = INPUT_I[2], eps2 = INPUT_I[3];
        const float xj = INPUT_J[0], yj = INPUT_J[1], zj = INPUT_J[2], mj = INPUT_J[3];
        const float dx = xj - xi, dy = yj - yi, dz = zj - zi;
        const bool coincident = (dx == 0.0f && dy == 0.0f && dz == 0.0f);                   // reading R1, branch-free:
        const float dx2 = dx * dx, dy2 = dy * dy, dz2 = dz * dz;
        const float r2 = (dx2 + dy2) + (dz2 + eps2);
        const float r1i = coincident ? 0.0f : pipeline_rsqrt(r2);                           // PAPER.md:465; r1i = 0 => the pair adds 0
        const float r2i = r1i * r1i;
        const float r3i = r2i * r1i;
        const float mr3i = mj * r3i;
        OUTPUT[0] += mr3i * dx;
        OUTPUT[1] += mr3i * dy;
        OUTPUT[2] += mr3i * dz;
    }
};

// Fig. A.2 / A.4: IDIM 6 = (x, v), JDIM 7 = (x, v, m), FDIM 7 = (a, jerk, pot);
// eps2 is the listing's constant 1/(256*256).
struct PipelineForceJerkPotA4 {
    static constexpr int IDIM = 6, JDIM = 7, FDIM = 7;
    static __device__ __forceinline__ void pair(const float* INPUT_I, const float* INPUT_J, float* OUTPUT) {
        const float eps2 = 1.0f / (256.0f * 256.0f);
        const float dx_0 = INPUT_J[0] - INPUT_I[0], dx_1 = INPUT_J[1] - INPUT_I[1], dx_2 = INPUT_J[2] - INPUT_I[2];
        const bool coincident = (dx_0 == 0.0f && dx_1 == 0.0f && dx_2 == 0.0f);             // reading R1, branch-free:
        const float mj = INPUT_J[6];
        const float r2 = coincident ? 1.0f : dx_0 * dx_0 + dx_1 * dx_1 + dx_2 * dx_2 + eps2;   // PAPER.md:506-509 (r2 = 1: finite)
        const float r1i = coincident ? 0.0f : pipeline_rsqrt(r2);                           // PAPER.md:510; r1i = 0 => the pair adds 0
        const float r2i = r1i * r1i, r3i = r1i * r2i, r5i = r2i * r3i;
        const float mr5i = mj * r5i, mf = mr5i * r2, pot = mf * r2;
        const float dv_0 = INPUT_J[3] - INPUT_I[3], dv_1 = INPUT_J[4] - INPUT_I[4], dv_2 = INPUT_J[5] - INPUT_I[5];
        const float mf3a = 3.0f * mr5i * (dx_0 * dv_0 + dx_1 * dv_1 + dx_2 * dv_2);
        OUTPUT[0] += mf * dx_0;
        OUTPUT[1] += mf * dx_1;
        OUTPUT[2] += mf * dx_2;
        OUTPUT[3] += mf * dv_0 - mf3a * dx_0;
        OUTPUT[4] += mf * dv_1 - mf3a * dx_1;
        OUTPUT[5] += mf * dv_2 - mf3a * dx_2;
        OUTPUT[6] -= pot;
    }
};

// A central force other than gravity (section 4.5: "van der Waals molecular interactions"; no formula in
// the paper -- DESIGN.md reading R19): 12-6 Lennard-Jones with Lorentz-Berthelot mixing, all pairs, no cut-off.
// IDIM 5 = (x, y, z, sigma_i / 2, sqrt(eps_i)), JDIM 5 likewise, FDIM 4 = (Fx, Fy, Fz, U): force ON i, pair energies of i.
struct PipelineLennardJones {
    static constexpr int IDIM = 5, JDIM = 5, FDIM = 4;
    static __device__ __forceinline__ void pair(const float* INPUT_I, const float* INPUT_J, float* OUTPUT) {
        const float dx = INPUT_J[0] - INPUT_I[0], dy = INPUT_J[1] - INPUT_I[1], dz = INPUT_J[2] - INPUT_I[2];
        const float r2 = dx * dx + dy * dy + dz * dz;
        const float r1i = (r2 == 0.0f) ? 0.0f : pipeline_rsqrt(r2);    // reading R1, branch-free: r1i = 0 => the pair adds 0
        const float r2i = r1i * r1i;
        const float sigma = INPUT_I[3] + INPUT_J[3], eps = INPUT_I[4] * INPUT_J[4];         // Lorentz-Berthelot
        const float s2 = sigma * sigma * r2i, s6 = s2 * s2 * s2;
        const float es6 = eps * s6;
        const float f = 24.0f * es6 * (2.0f * s6 - 1.0f) * r2i;        // 24 eps (2 s^12 - s^6) / r^2
        OUTPUT[0] -= f * dx;
        OUTPUT[1] -= f * dy;
        OUTPUT[2] -= f * dz;
        OUTPUT[3] += 4.0f * es6 * (s6 - 1.0f);                         // 4 eps (s^12 - s^6)
    }
};

}  // namespace nb
