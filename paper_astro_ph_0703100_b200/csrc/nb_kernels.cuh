// nb_kernels.cuh -- sm_100a device code for the all-pairs softened gravity path.
//
// Rows of SURVEY.md section 8(a) implemented here (citations: PAPER.md by line):
//   a1  j-pack            nb_pack_pairs_kernel     Fig. A.1 packing loop
//   a2  j-tile staging    TMA bulk copy + mbarrier ring in nb_force_kernel   step (d) J-PACKING
//   a3  i-load            prologue of nb_force_kernel                        step (e)
//   a4  pair interaction  pair_body()                                        step (h); Eq. (1); Fig. A.3 PAPER.md:458-471;
//                                                                            potential Fig. A.4
//   a5  two-level sum     per-tile partial -> running total                  steps (f),(g),(i); Eq. (2)
//   a6  epilogue          end of nb_force_kernel / nb_reduce_kernel          step (i)
//   a7  j-split + reduce  WJ (warps) and S (CTAs) split, fixed-order sums    (paper analogue: force-memory round trips)
//
// Layout of the packed j-array ("pair records", 32 B each, 128-B aligned array):
//     record p = { x[2p], x[2p+1], y[2p], y[2p+1],   z[2p], z[2p+1], m[2p], m[2p+1] }
// so that one LDS.128 yields two 64-bit operands for the packed FP32 instructions
// (add/mul/fma.f32x2 -> SASS FADD2/FMUL2/FFMA2): the two halves of every packed operand are two
// consecutive j-particles interacting with the same i-particle.
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

// ---------------------------------------------------------------- a1: j-pack
// One thread per pair record.  Particles beyond n_j (padding up to a multiple of 8) take the
// position of the last real particle and mass 0, so they contribute exactly nothing.
__global__ void __launch_bounds__(256) nb_pack_pairs_kernel(const float* __restrict__ x_j, const float* __restrict__ m_j,
                                                            int n_j, int n_pairs_padded, float4* __restrict__ jp) {
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs_padded) return;
    int j0 = 2 * p, j1 = 2 * p + 1;
    int c0 = min(j0, n_j - 1), c1 = min(j1, n_j - 1);
    float x0 = x_j[3 * c0 + 0], y0 = x_j[3 * c0 + 1], z0 = x_j[3 * c0 + 2];
    float x1 = x_j[3 * c1 + 0], y1 = x_j[3 * c1 + 1], z1 = x_j[3 * c1 + 2];
    float m0 = (j0 < n_j) ? m_j[c0] : 0.0f;
    float m1 = (j1 < n_j) ? m_j[c1] : 0.0f;
    jp[2 * p + 0] = make_float4(x0, x1, y0, y1);
    jp[2 * p + 1] = make_float4(z0, z1, m0, m1);
}

// ---------------------------------------------------------------- a4: one i-particle x one j-pair
// 13 packed FP32-pipe instructions (3 FADD2, 3 FFMA2, 3 FMUL2, 3 FFMA2, 1 FADD2) + 2 MUFU.RSQ
// + the coincidence mask on the ALU pipe.  nxi = (-x_i, -x_i) etc., so d = r_j - r_i.
template <bool EXACT_MASK>
__device__ __forceinline__ void pair_body(u64 xj, u64 yj, u64 zj, u64 mj, u64 nxi, u64 nyi, u64 nzi, u64 eps2_2,
                                          float eps2, u64& ax, u64& ay, u64& az, u64& ph) {
    const u64 dx = add2(xj, nxi);                    // dx = xj - xi
    const u64 dy = add2(yj, nyi);
    const u64 dz = add2(zj, nzi);
    u64 r2 = fma2(dx, dx, eps2_2);                   // r2 = dx2+dy2+dz2+eps2 PAPER.md:464
    r2 = fma2(dy, dy, r2);
    r2 = fma2(dz, dz, r2);
    float r2a, r2b;
    unpack2(r2, r2a, r2b);
    const float inf = __int_as_float(0x7f800000);
    if (EXACT_MASK) {
        // coincident <=> all three differences are exactly +0 (x - x rounds to +0)
        float dxa, dxb, dya, dyb, dza, dzb;
        unpack2(dx, dxa, dxb); unpack2(dy, dya, dyb); unpack2(dz, dza, dzb);
        const uint32_t ta = __float_as_uint(dxa) | __float_as_uint(dya) | __float_as_uint(dza);
        const uint32_t tb = __float_as_uint(dxb) | __float_as_uint(dyb) | __float_as_uint(dzb);
        r2a = (ta == 0u) ? inf : r2a;                // rsqrt(+inf) = +0 -> the pair adds exactly 0
        r2b = (tb == 0u) ? inf : r2b;
    } else {
        r2a = (r2a == eps2) ? inf : r2a;
        r2b = (r2b == eps2) ? inf : r2b;
    }
    const u64 u = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));   // r1i = 1/sqrt(r2)
    const u64 u2 = mul2(u, u);                       // r2i
    const u64 mu = mul2(mj, u);                      // pot = mj * r1i
    const u64 mu3 = mul2(mu, u2);                    // mr3i
    ax = fma2(mu3, dx, ax);                          // OUTPUT[0..2] += mr3i*d PAPER.md:469-471
    ay = fma2(mu3, dy, ay);
    az = fma2(mu3, dz, az);
    ph = add2(ph, mu);                               // OUTPUT[6] -= pot (sign applied at the end) PAPER.md:552
}

struct ForceArgs {
    const float* x_i;      // [n_i][3]
    const ulonglong2* jp;  // packed pair records, 2 x 16 B per pair
    float* acc;            // [n_i][3]
    float* pot;            // [n_i] or nullptr
    double4* partial;      // [S][n_i] when S > 1
    int n_i;
    int n_units;           // padded pairs / 4
    int S;
    float eps2;
};

// ---------------------------------------------------------------- a2..a7: the force kernel
// CTA = 8 warps = WI (along i) x WJ (along j).  A CTA owns 32*K*WI i-particles (K per thread, in
// registers) and the S-th part (blockIdx.y) of the j-range, which is cut again into WJ sub-ranges.
// Each sub-range is streamed through its own shared-memory ring by 1-D TMA bulk copies issued by
// lane 0 of the group's first warp; "full" mbarriers count bytes, "empty" mbarriers count the WI
// consuming warps.
template <int K, int WI, int WJ, int TP, int STAGES, bool EXACT_MASK>
__global__ void __launch_bounds__(32 * WI * WJ, 1) nb_force_kernel(const ForceArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int RING_BYTES = STAGES * TP * 32;
    unsigned char* rings = smem_raw;                                   // [WJ][STAGES][TP*32]
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + WJ * RING_BYTES);   // full[WJ][STAGES], empty[WJ][STAGES]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wi = warp % WI, wj = warp / WI;
    const bool producer = (wi == 0) && (lane == 0);

    const uint32_t ring = smem_u32(rings + wj * RING_BYTES);
    const uint32_t full0 = smem_u32(bars + wj * STAGES);
    const uint32_t empty0 = smem_u32(bars + (WJ + wj) * STAGES);

    if (producer) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, WI);
        }
        mbar_fence_init();
    }

    // j sub-range of this warp group, in units of 4 pairs
    const long long G = (long long)a.S * WJ;
    const long long g = (long long)blockIdx.y * WJ + wj;
    const int u_begin = (int)((long long)a.n_units * g / G);
    const int u_end = (int)((long long)a.n_units * (g + 1) / G);
    const int n_sub = (u_end - u_begin) * 4;                           // pairs
    const int n_tiles = (n_sub + TP - 1) / TP;
    const unsigned char* src = reinterpret_cast<const unsigned char*>(a.jp) + (size_t)u_begin * 128;

    // a3: i-particles of this thread (clamped loads; stores are guarded)
    const int i_base = blockIdx.x * (32 * K * WI) + wi * 32 + lane;
    u64 nxi[K], nyi[K], nzi[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int i = min(i_base + k * 32 * WI, a.n_i - 1);
        const float x = a.x_i[3 * i + 0], y = a.x_i[3 * i + 1], z = a.x_i[3 * i + 2];
        nxi[k] = pack2(-x, -x); nyi[k] = pack2(-y, -y); nzi[k] = pack2(-z, -z);
    }
    const float eps2 = a.eps2;
    const u64 eps2_2 = pack2(eps2, eps2);

    __syncthreads();                                                   // barriers initialised

    if (producer) {
        const int pre = n_tiles < STAGES ? n_tiles : STAGES;
        for (int t = 0; t < pre; ++t) {
            const uint32_t bytes = (uint32_t)min(TP, n_sub - t * TP) * 32u;
            mbar_expect_tx(full0 + 8 * t, bytes);
            tma_load_1d(ring + t * TP * 32, src + (size_t)t * TP * 32, bytes, full0 + 8 * t);
        }
    }

    double run[K][4];                                                  // running totals (outer level of Eq. (2))
#pragma unroll
    for (int k = 0; k < K; ++k) { run[k][0] = run[k][1] = run[k][2] = run[k][3] = 0.0; }

    for (int t = 0; t < n_tiles; ++t) {
        const int slot = t % STAGES;
        const uint32_t parity = (uint32_t)(t / STAGES) & 1u;
        mbar_wait(full0 + 8 * slot, parity);

        const int np = min(TP, n_sub - t * TP);                        // multiple of 4
        const ulonglong2* sp = reinterpret_cast<const ulonglong2*>(rings + wj * RING_BYTES + slot * TP * 32);

        u64 pax[K], pay[K], paz[K], pph[K];                            // tile partial sums, started from zero (Eq. (2))
#pragma unroll
        for (int k = 0; k < K; ++k) { pax[k] = 0ull; pay[k] = 0ull; paz[k] = 0ull; pph[k] = 0ull; }

#pragma unroll 4
        for (int p = 0; p < np; ++p) {
            const ulonglong2 A = sp[2 * p + 0];                        // broadcast LDS.128: x0 x1 | y0 y1
            const ulonglong2 B = sp[2 * p + 1];                        //                    z0 z1 | m0 m1
#pragma unroll
            for (int k = 0; k < K; ++k)
                pair_body<EXACT_MASK>(A.x, A.y, B.x, B.y, nxi[k], nyi[k], nzi[k], eps2_2, eps2, pax[k], pay[k], paz[k], pph[k]);
        }

        // a5: tile partial -> running total
#pragma unroll
        for (int k = 0; k < K; ++k) {
            float lo, hi;
            unpack2(pax[k], lo, hi); run[k][0] += (double)(lo + hi);
            unpack2(pay[k], lo, hi); run[k][1] += (double)(lo + hi);
            unpack2(paz[k], lo, hi); run[k][2] += (double)(lo + hi);
            unpack2(pph[k], lo, hi); run[k][3] += (double)(lo + hi);
        }

        // release the slot; the producer refills it with tile t' + STAGES.  With several consumer
        // warps the refill trails by one tile so that the producer rarely waits for a slower warp.
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
        if (producer) {
            const int tt = (WI > 1) ? t - 1 : t;
            if (tt >= 0 && tt + STAGES < n_tiles) {
                const int rs = tt % STAGES;
                mbar_wait(empty0 + 8 * rs, (uint32_t)(tt / STAGES) & 1u);
                const int tn = tt + STAGES;
                const uint32_t bytes = (uint32_t)min(TP, n_sub - tn * TP) * 32u;
                mbar_expect_tx(full0 + 8 * rs, bytes);
                tma_load_1d(ring + rs * TP * 32, src + (size_t)tn * TP * 32, bytes, full0 + 8 * rs);
            }
        }
        __syncwarp();
    }

    // a7 (intra-CTA): fixed-order sum over the WJ warp groups through shared memory
    if (WJ > 1) {
        __syncthreads();                                               // all rings drained; reuse the memory
        double* red = reinterpret_cast<double*>(smem_raw);             // [WJ][K][4][WI*32]
        const int tig = wi * 32 + lane;
#pragma unroll
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int c = 0; c < 4; ++c) red[((wj * K + k) * 4 + c) * (WI * 32) + tig] = run[k][c];
        __syncthreads();
        if (wj != 0) return;
#pragma unroll
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                double s = red[((0 * K + k) * 4 + c) * (WI * 32) + tig];
#pragma unroll
                for (int w = 1; w < WJ; ++w) s += red[((w * K + k) * 4 + c) * (WI * 32) + tig];
                run[k][c] = s;
            }
    }

    // a6: epilogue
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int i = i_base + k * 32 * WI;
        if (i >= a.n_i) continue;
        if (a.S == 1) {
            a.acc[3 * i + 0] = (float)run[k][0];
            a.acc[3 * i + 1] = (float)run[k][1];
            a.acc[3 * i + 2] = (float)run[k][2];
            if (a.pot) a.pot[i] = -(float)run[k][3];
        } else {
            a.partial[(size_t)blockIdx.y * a.n_i + i] = make_double4(run[k][0], run[k][1], run[k][2], run[k][3]);
        }
    }
}

// a7 (inter-CTA): second pass, fixed-order sum over the S chunk partials
__global__ void __launch_bounds__(128) nb_reduce_kernel(const double4* __restrict__ partial, int n_i, int S,
                                                        float* __restrict__ acc, float* __restrict__ pot) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_i) return;
    double4 s = partial[i];
    for (int c = 1; c < S; ++c) {
        const double4 v = partial[(size_t)c * n_i + i];
        s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
    }
    acc[3 * i + 0] = (float)s.x;
    acc[3 * i + 1] = (float)s.y;
    acc[3 * i + 2] = (float)s.z;
    if (pot) pot[i] = -(float)s.w;
}

// ---------------------------------------------------------------- a8: leapfrog O(N) kernels
// kick:  v += a * h        (h = dt/2)
__global__ void __launch_bounds__(256) nb_kick_kernel(float* __restrict__ v, const float* __restrict__ acc, int n3, float h) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n3) v[k] = fmaf(acc[k], h, v[k]);
}
// closing half-kick of step s fused with the opening half-kick and drift of step s+1:
//   v += a*h;  [v += a*h;]  x += v*dt      (two separately rounded kicks, exactly as if unfused)
template <bool TWO_KICKS>
__global__ void __launch_bounds__(256) nb_kick_drift_kernel(float* __restrict__ x, float* __restrict__ v,
                                                            const float* __restrict__ acc, int n3, float h, float dt) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n3) return;
    const float aa = acc[k];
    float vv = fmaf(aa, h, v[k]);
    if (TWO_KICKS) vv = fmaf(aa, h, vv);
    v[k] = vv;
    x[k] = fmaf(vv, dt, x[k]);
}

}  // namespace nb
