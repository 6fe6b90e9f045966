// nb_packed.cuh -- inline device helpers shared by the kernels and by user pipelines (nb_pipeline.cuh): packed FP32 (f32x2) arithmetic, mbarrier / TMA bulk copy,
// and the coincident-pair conventions (reading R1).  Inline functions only: safe in several translation units.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nb {

typedef unsigned long long u64;

// ---------------------------------------------------------------- packed FP32 helpers
__device__ __forceinline__ u64 pack2(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 d;
    asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b) {
    u64 d;
    asm("sub.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 d;
    asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 d;
    asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---------------------------------------------------------------- mbarrier / TMA bulk copy
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n"
            "  .reg .pred p;\n"
            "  mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "  selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// ---------------------------------------------------------------- coincident pairs (reading R1)
enum { MASK_EXACT = 0, MASK_NONE = 2 };

// -x_i as the kernels hold it: +0 for a zero or subnormal coordinate (add.ftz reads a subnormal as zero), so that a
// difference x_j + (-x_i) that is zero is always +0 -- (-0) + (-0) = -0 cannot arise -- and the bitwise test of
// MASK_EXACT sees every coincident pair, whatever the signs of the zeros involved.
__device__ __forceinline__ float neg_canon(float x) { return (fabsf(x) < 1.17549435e-38f) ? 0.0f : -x; }

// canonical position bits (subnormals and -0 -> +0, as add.ftz sees them) and their hash: the coincidence pre-pass of
// large calls (nb_kernels.cuh) (kept with the packed helpers: inline, several translation units)
__device__ __forceinline__ uint32_t coin_canon(float v) {
    return (fabsf(v) < 1.17549435e-38f) ? 0u : __float_as_uint(v);
}
__device__ __forceinline__ uint32_t coin_hash(uint32_t a, uint32_t b, uint32_t c) {
    uint64_t h = (uint64_t)a * 0x9E3779B97F4A7C15ull;
    h ^= (uint64_t)b * 0xC2B2AE3D27D4EB4Full + (h >> 29);
    h ^= (uint64_t)c * 0x165667B19E3779F9ull + (h << 17);
    h ^= h >> 32;
    h *= 0xD6E8FEB86659FD93ull;
    return (uint32_t)(h >> 32);
}

// ---------------------------------------------------------------- Bloom filter of a warp's i-positions (block-level coincidence test)
// MODE_BLOOM: 2^16 filter bits (8 KB) per group of warps that hold the same i-particles, two bits per position.
// The key is computed on the coordinates as the loop sees them (x + 0 under add.ftz: -0 and subnormals become +0),
// so two positions the masked loop calls coincident always have the same key: no false negatives.
constexpr int kBloomWords = 2048;
__device__ __forceinline__ uint32_t bloom_key(float x, float y, float z) {
    float cx, cy, cz;
    asm("add.ftz.f32 %0, %1, 0f00000000;" : "=f"(cx) : "f"(x));
    asm("add.ftz.f32 %0, %1, 0f00000000;" : "=f"(cy) : "f"(y));
    asm("add.ftz.f32 %0, %1, 0f00000000;" : "=f"(cz) : "f"(z));
    uint32_t h = __float_as_uint(cx) * 0x9E3779B1u;
    h = __float_as_uint(cy) * 0x85EBCA77u + h;
    h = __float_as_uint(cz) * 0xC2B2AE3Du + (h ^ (h >> 15));
    h ^= h >> 16;
    return h * 0x2C1B3C6Du;
}
__device__ __forceinline__ void bloom_set(uint32_t* filt, uint32_t h) {
    atomicOr(filt + (h >> 21), 1u << ((h >> 16) & 31u));
    atomicOr(filt + ((h >> 5) & 2047u), 1u << (h & 31u));
}
__device__ __forceinline__ bool bloom_test(const uint32_t* filt, uint32_t h) {
    return ((filt[h >> 21] >> ((h >> 16) & 31u)) & (filt[(h >> 5) & 2047u] >> (h & 31u)) & 1u) != 0u;
}

}  // namespace nb
