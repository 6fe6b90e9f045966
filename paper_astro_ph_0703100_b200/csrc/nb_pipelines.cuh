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
    // The same statements for two i-records at once (nb_pipeline.cuh, packed path): I2[c] = (rec0[c], rec1[c]).
    static constexpr bool kPacked = true, kCoincidentRule = true;
    static __device__ __forceinline__ void prep_i(float* rec) {        // positions are held as -x, zeros canonicalised (reading R1)
        rec[0] = neg_canon(rec[0]); rec[1] = neg_canon(rec[1]); rec[2] = neg_canon(rec[2]);
    }
    template <bool MASKED>
    static __device__ __forceinline__ void pair2(const u64* I2, const float* INPUT_J, u64* OUT2) {
        const float xj = INPUT_J[0], yj = INPUT_J[1], zj = INPUT_J[2], mj = INPUT_J[3];
        const u64 dx = add2(pack2(xj, xj), I2[0]), dy = add2(pack2(yj, yj), I2[1]), dz = add2(pack2(zj, zj), I2[2]);
        u64 r2 = fma2(dx, dx, I2[3]);                                                      // PAPER.md:461-464 (any order: reading R6)
        r2 = fma2(dy, dy, r2);
        r2 = fma2(dz, dz, r2);
        float ra, rb;
        unpack2(r2, ra, rb);
        if (MASKED) {
            float a0, a1, b0, b1, c0, c1;
            unpack2(dx, a0, a1); unpack2(dy, b0, b1); unpack2(dz, c0, c1);
            const uint32_t ta = __float_as_uint(a0) | __float_as_uint(b0) | __float_as_uint(c0);
            const uint32_t tb = __float_as_uint(a1) | __float_as_uint(b1) | __float_as_uint(c1);
            ra = (ta == 0u) ? __int_as_float(0x7f800000) : ra;         // rsqrt(+inf) = +0: the pair adds 0
            rb = (tb == 0u) ? __int_as_float(0x7f800000) : rb;
        }
        const u64 r1i = pack2(pipeline_rsqrt(ra), pipeline_rsqrt(rb));
        const u64 r2i = mul2(r1i, r1i);
        const u64 mr1i = mul2(pack2(mj, mj), r1i);
        const u64 mr3i = mul2(mr1i, r2i);
        OUT2[0] = fma2(mr3i, dx, OUT2[0]);
        OUT2[1] = fma2(mr3i, dy, OUT2[1]);
        OUT2[2] = fma2(mr3i, dz, OUT2[2]);
    }
    static __device__ __forceinline__ void finish(const double* sum, float* OUTPUT) {
        OUTPUT[0] = (float)sum[0]; OUTPUT[1] = (float)sum[1]; OUTPUT[2] = (float)sum[2];
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
    // Packed form: the listing's statements for two i-records at once; d = x_j - x_i and dv = v_j - v_i are formed through
    // -x_i (canonicalised, reading R1) and -v_i; pot is summed with its sign applied at the end.
    static constexpr bool kPacked = true, kCoincidentRule = true;
    static __device__ __forceinline__ void prep_i(float* rec) {        // -x canonicalised, -v
        rec[0] = neg_canon(rec[0]); rec[1] = neg_canon(rec[1]); rec[2] = neg_canon(rec[2]);
        rec[3] = -rec[3]; rec[4] = -rec[4]; rec[5] = -rec[5];
    }
    template <bool MASKED>
    static __device__ __forceinline__ void pair2(const u64* I2, const float* INPUT_J, u64* OUT2) {
        const float e2 = 1.0f / (256.0f * 256.0f);
        const u64 dx0 = add2(pack2(INPUT_J[0], INPUT_J[0]), I2[0]), dx1 = add2(pack2(INPUT_J[1], INPUT_J[1]), I2[1]),
                  dx2 = add2(pack2(INPUT_J[2], INPUT_J[2]), I2[2]);
        u64 r2 = fma2(dx0, dx0, pack2(e2, e2));
        r2 = fma2(dx1, dx1, r2);
        r2 = fma2(dx2, dx2, r2);
        float ra, rb;
        unpack2(r2, ra, rb);
        if (MASKED) {
            float a0, a1, b0, b1, c0, c1;
            unpack2(dx0, a0, a1); unpack2(dx1, b0, b1); unpack2(dx2, c0, c1);
            const uint32_t ta = __float_as_uint(a0) | __float_as_uint(b0) | __float_as_uint(c0);
            const uint32_t tb = __float_as_uint(a1) | __float_as_uint(b1) | __float_as_uint(c1);
            ra = (ta == 0u) ? __int_as_float(0x7f800000) : ra;         // r1i = +0: the pair adds 0
            rb = (tb == 0u) ? __int_as_float(0x7f800000) : rb;
        }
        const u64 r1i = pack2(pipeline_rsqrt(ra), pipeline_rsqrt(rb));
        const u64 r2i = mul2(r1i, r1i);
        const u64 pot = mul2(pack2(INPUT_J[6], INPUT_J[6]), r1i);                           // pot = mj r1i
        const u64 mf = mul2(pot, r2i);                                                      // mf = mj r3i
        const u64 dv0 = add2(pack2(INPUT_J[3], INPUT_J[3]), I2[3]), dv1 = add2(pack2(INPUT_J[4], INPUT_J[4]), I2[4]),
                  dv2 = add2(pack2(INPUT_J[5], INPUT_J[5]), I2[5]);
        u64 xv = mul2(dx0, dv0);
        xv = fma2(dx1, dv1, xv);
        xv = fma2(dx2, dv2, xv);
        const u64 nmf3a = mul2(mul2(mf, r2i), mul2(xv, pack2(-3.0f, -3.0f)));               // -3 mr5i (dx.dv)
        OUT2[0] = fma2(mf, dx0, OUT2[0]);
        OUT2[1] = fma2(mf, dx1, OUT2[1]);
        OUT2[2] = fma2(mf, dx2, OUT2[2]);
        OUT2[3] = fma2(nmf3a, dx0, fma2(mf, dv0, OUT2[3]));
        OUT2[4] = fma2(nmf3a, dx1, fma2(mf, dv1, OUT2[4]));
        OUT2[5] = fma2(nmf3a, dx2, fma2(mf, dv2, OUT2[5]));
        OUT2[6] = add2(OUT2[6], pot);                                                       // sign at the end
    }
    static __device__ __forceinline__ void finish(const double* sum, float* OUTPUT) {
#pragma unroll
        for (int c = 0; c < 6; ++c) OUTPUT[c] = (float)sum[c];
        OUTPUT[6] = -(float)sum[6];
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
    // Packed form.  d = r_j - r_i is held through -r_i; the force on i is -f d: accumulate +f d and flip the sign at the end.
    static constexpr bool kPacked = true, kCoincidentRule = true;
    static __device__ __forceinline__ void prep_i(float* rec) {
        rec[0] = neg_canon(rec[0]); rec[1] = neg_canon(rec[1]); rec[2] = neg_canon(rec[2]);
    }
    template <bool MASKED>
    static __device__ __forceinline__ void pair2(const u64* I2, const float* INPUT_J, u64* OUT2) {
        const u64 dx = add2(pack2(INPUT_J[0], INPUT_J[0]), I2[0]), dy = add2(pack2(INPUT_J[1], INPUT_J[1]), I2[1]),
                  dz = add2(pack2(INPUT_J[2], INPUT_J[2]), I2[2]);
        u64 r2 = mul2(dx, dx);
        r2 = fma2(dy, dy, r2);
        r2 = fma2(dz, dz, r2);
        float ra, rb;
        unpack2(r2, ra, rb);
        if (MASKED) {                                                  // r2 == 0 (coincident, or closer than 1e-19): r1i = 0
            ra = (ra == 0.0f) ? __int_as_float(0x7f800000) : ra;
            rb = (rb == 0.0f) ? __int_as_float(0x7f800000) : rb;
        }
        const u64 r1i = pack2(pipeline_rsqrt(ra), pipeline_rsqrt(rb));
        const u64 r2i = mul2(r1i, r1i);
        const u64 sigma = add2(pack2(INPUT_J[3], INPUT_J[3]), I2[3]);                       // Lorentz-Berthelot
        const u64 eps = mul2(pack2(INPUT_J[4], INPUT_J[4]), I2[4]);
        const u64 s2 = mul2(mul2(sigma, sigma), r2i);
        const u64 s6 = mul2(mul2(s2, s2), s2);
        const u64 es6 = mul2(eps, s6);
        const u64 f = mul2(mul2(es6, pack2(24.0f, 24.0f)), mul2(fma2(s6, pack2(2.0f, 2.0f), pack2(-1.0f, -1.0f)), r2i));
        OUT2[0] = fma2(f, dx, OUT2[0]);
        OUT2[1] = fma2(f, dy, OUT2[1]);
        OUT2[2] = fma2(f, dz, OUT2[2]);
        OUT2[3] = fma2(mul2(es6, pack2(4.0f, 4.0f)), add2(s6, pack2(-1.0f, -1.0f)), OUT2[3]);
    }
    static __device__ __forceinline__ void finish(const double* sum, float* OUTPUT) {
        OUTPUT[0] = -(float)sum[0]; OUTPUT[1] = -(float)sum[1]; OUTPUT[2] = -(float)sum[2]; OUTPUT[3] = (float)sum[3];
    }
};

}  // namespace nb
