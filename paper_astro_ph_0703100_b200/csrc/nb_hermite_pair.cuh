// nb_hermite_pair.cuh -- the force + jerk + potential pair arithmetic of Fig. A.4 on packed f32x2
// operands, shared by nb_hermite_kernel (nb_hermite.cuh: the two halves are two i-particles, the j-particle is broadcast)
// and nb_small_hermite_kernel (nb_small_hermite.cuh: the two halves are two consecutive j-particles, the i-particle is
// broadcast).  Inline device code only: includable from several translation units.
#pragma once
#include <stdint.h>

#include "../../include/nb_packed.cuh"

namespace nb {

constexpr int kHermiteAcc = 10;   // ax ay az | j1x j1y j1z | j2x j2y j2z | phi

// PHI = false: the caller does not want the potential: 26 FP32-pipe instructions per pair.
template <bool MASKED, bool PHI = true>
__device__ __forceinline__ void hermite_pair(u64 xj, u64 yj, u64 zj, u64 mj, u64 vxj, u64 vyj, u64 vzj,
                                             u64 nxi, u64 nyi, u64 nzi, u64 nvxi, u64 nvyi, u64 nvzi, u64 eps2_2,
                                             u64 (&s)[kHermiteAcc]) {
    const u64 dx = add2(xj, nxi);                    // dx = xj - xi
    const u64 dy = add2(yj, nyi);
    const u64 dz = add2(zj, nzi);
    u64 r2 = fma2(dx, dx, eps2_2);                   // r2 = dx.dx + eps2
    r2 = fma2(dy, dy, r2);
    r2 = fma2(dz, dz, r2);
    float r2a, r2b;
    unpack2(r2, r2a, r2b);
    if (MASKED) {
        const float inf = __int_as_float(0x7f800000);
        float dxa, dxb, dya, dyb, dza, dzb;
        unpack2(dx, dxa, dxb); unpack2(dy, dya, dyb); unpack2(dz, dza, dzb);
        const uint32_t ta = __float_as_uint(dxa) | __float_as_uint(dya) | __float_as_uint(dza);
        const uint32_t tb = __float_as_uint(dxb) | __float_as_uint(dyb) | __float_as_uint(dzb);
        r2a = (ta == 0u) ? inf : r2a;                // rsqrt(+inf) = +0 -> every term of the pair is exactly 0
        r2b = (tb == 0u) ? inf : r2b;
    }
    const u64 u = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));   // r1i
    const u64 u2 = mul2(u, u);                       // r2i
    const u64 mu = mul2(mj, u);                      // pot = mj r1i
    const u64 mu3 = mul2(mu, u2);                    // mf  = mj r3i
    const u64 dvx = add2(vxj, nvxi);                 // dv = vj - vi
    const u64 dvy = add2(vyj, nvyi);
    const u64 dvz = add2(vzj, nvzi);
    u64 xv = mul2(dx, dvx);                          // xv0 + xv1 + xv2
    xv = fma2(dy, dvy, xv);
    xv = fma2(dz, dvz, xv);
    const u64 q = mul2(u2, xv);
    const u64 w = mul2(mu3, q);                      // mr5i (d.dv)   (mf3a / 3)
    s[0] = fma2(mu3, dx, s[0]);                      // OUTPUT[0..2] += fx
    s[1] = fma2(mu3, dy, s[1]);
    s[2] = fma2(mu3, dz, s[2]);
    s[3] = fma2(mu3, dvx, s[3]);                     // jk1 = mf dv
    s[4] = fma2(mu3, dvy, s[4]);
    s[5] = fma2(mu3, dvz, s[5]);
    s[6] = fma2(w, dx, s[6]);                        // jk2 / 3 = mr5i (d.dv) d
    s[7] = fma2(w, dy, s[7]);
    s[8] = fma2(w, dz, s[8]);
    if (PHI) s[9] = add2(s[9], mu);                  // OUTPUT[6] -= pot (sign at the end)
}

}  // namespace nb
