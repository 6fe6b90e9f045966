// nb_hermite.cuh -- sm_100a device code for row f1: force + jerk + potential for the 4th-order
// Hermite scheme, the paper's second pipeline description (Fig. A.2 PAPER.md:397-428,
// Fig. A.4):
//
//     a_i    =  sum_j m_j d / r^3                          d = r_j - r_i,  r^2 = d.d + eps^2
//     jerk_i =  sum_j m_j [ dv / r^3 - 3 (d.dv) d / r^5 ]  dv = v_j - v_i
//     phi_i  = -sum_j m_j / r
//
// Same structure as nb_force_kernel (nb_kernels.cuh): i stationary in registers as packed pairs,
// j streamed through a TMA + mbarrier ring, Eq. (2) two-level sums (FP32 partials over <= 256 j,
// FP64 running totals), WJ x S j-split with fixed-order reductions.  Differences:
//   - j record = 32 bytes (x, y, z, m | vx, vy, vz, 0): the paper's [n_j][JDIM = 7] row
//     padded to two LDS.128;
//   - 10 accumulators per i-particle: a (3), J1 = sum mf dv (3), J2 = sum mr5i (d.dv) d (3), phi;
//     jerk = J1 - 3 J2 is formed once, in FP64, in the epilogue (jk = jk1 - jk2 with
//     mf3a = 3 mr5i (xv0+xv1+xv2)) -- the factor 3 leaves the hot loop;
//   - per pair 27 FP32-pipe instructions + 1 MUFU.RSQ:
//       3 FADD (d)  3 FFMA (r2)  3 FMUL (u2, m u, m u^3)  3 FADD (dv)  1 FMUL + 2 FFMA (d.dv)
//       2 FMUL (u2 (d.dv), m u^5 (d.dv))  3 FFMA (a)  3 FFMA (J1)  3 FFMA (J2)  1 FADD (phi).
// Coincident pairs (all three POSITION differences exactly zero, reading R1) add nothing:
// MODE_EXACT masks every pair; MODE_BLOOM tests every 256-j block against a filter of the warp's i-positions;
// MODE_LIST uses the coincidence lists of the pre-pass (all three: nb_kernels.cuh)
// and masks only the listed j-segments.  An unmasked coincident pair would add m dv / eps^3 to the
// jerk, so unlike the plain force there is no speculative mode here.
#pragma once
#include <math_constants.h>
#include "nb_kernels.cuh"
#include "nb_hermite_pair.cuh"

namespace nb {

#ifndef NB_HERMITE_UNROLL
#define NB_HERMITE_UNROLL 2
#endif
constexpr int kHermiteUnroll = NB_HERMITE_UNROLL;   // j-particles per loop iteration (measured: 1 / 2 / 4)

// (x, y, z) || m || (vx, vy, vz) -> two float4 per j-particle
__global__ void __launch_bounds__(256) nb_pack_jv_kernel(const float* __restrict__ x_j, const float* __restrict__ v_j,
                                                         const float* __restrict__ m_j, int n_j, float4* __restrict__ jp) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_j) return;
    jp[2 * (size_t)j + 0] = make_float4(x_j[3 * (size_t)j + 0], x_j[3 * (size_t)j + 1], x_j[3 * (size_t)j + 2], m_j[j]);
    jp[2 * (size_t)j + 1] = make_float4(v_j[3 * (size_t)j + 0], v_j[3 * (size_t)j + 1], v_j[3 * (size_t)j + 2], 0.0f);
}

struct HermiteArgs {
    const float* x_i;      // [n_i][3]
    const float* v_i;      // [n_i][3]
    const float4* jp;      // [n_j][2] packed records
    float* acc;            // [n_i][3]
    float* jerk;           // [n_i][3]
    float* pot;            // [n_i] or nullptr
    double* partial;       // [S][n_i][10] when S > 1
    int* tickets;          // [tiles_i] zeroed counters: the last CTA of an i-tile makes the second pass; nullptr: separate launch
    const int* coin_lists;
    const int* coin_flag;
    int n_i;
    int n_j;
    int S;
    float eps2;
};

template <int K, bool MASKED, bool PHI = true>
__device__ __forceinline__ void hermite_sweep(const float4* __restrict__ sp, int np, const u64 (&ni)[K / 2][6], u64 eps2_2,
                                              u64 (&part)[K / 2][kHermiteAcc]) {
#pragma unroll
    for (int k = 0; k < K / 2; ++k)
#pragma unroll
        for (int c = 0; c < kHermiteAcc; ++c) part[k][c] = 0ull;
#pragma unroll kHermiteUnroll
    for (int j = 0; j < np; ++j) {
        const float4 P = sp[2 * j], V = sp[2 * j + 1];                 // two broadcast LDS.128
        const u64 xj = pack2(P.x, P.x), yj = pack2(P.y, P.y), zj = pack2(P.z, P.z), mj = pack2(P.w, P.w);
        const u64 vx = pack2(V.x, V.x), vy = pack2(V.y, V.y), vz = pack2(V.z, V.z);
#pragma unroll
        for (int k = 0; k < K / 2; ++k)
            hermite_pair<MASKED, PHI>(xj, yj, zj, mj, vx, vy, vz, ni[k][0], ni[k][1], ni[k][2], ni[k][3], ni[k][4], ni[k][5],
                                 eps2_2, part[k]);
    }
}

// CTA = 8 warps = WI x WJ, as nb_force_kernel.  TJ j-particles (32 B each) per ring stage.
template <int K, int WI, int WJ, int TJ, int STAGES, int MODE, bool PHI = true, int SUB = 256>
__global__ void __launch_bounds__(32 * WI * WJ, 1) nb_hermite_kernel(const HermiteArgs a) {
    static_assert(K % 2 == 0, "i-particles are held in pairs");
    static_assert(SUB == kCoinSeg, "coincidence segments are SUB j-particles");
    static_assert(MODE == MODE_EXACT || MODE == MODE_BLOOM || MODE == MODE_LIST, "masked everywhere, Bloom filter, or coincidence lists");
    constexpr bool FUSED = (MODE == MODE_EXACT);                       // can make the second pass itself (a.tickets)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int REC = 32;
    constexpr int RING_BYTES = STAGES * TJ * REC;
    unsigned char* rings = smem_raw;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + WJ * RING_BYTES);

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

    const long long G = (long long)a.S * WJ;
    const long long g = (long long)blockIdx.y * WJ + wj;
    const int j_begin = (int)((long long)a.n_j * g / G);
    const int j_end = (int)((long long)a.n_j * (g + 1) / G);
    const int n_sub = j_end - j_begin;
    const int n_tiles = (n_sub + TJ - 1) / TJ;
    const unsigned char* src = reinterpret_cast<const unsigned char*>(a.jp) + (size_t)j_begin * REC;

    const int i_base = blockIdx.x * (32 * K * WI) + wi * (32 * K) + lane;
    u64 ni[K / 2][6];                                                  // (-x, -y, -z, -vx, -vy, -vz) of each i-pair
#pragma unroll
    for (int k2 = 0; k2 < K / 2; ++k2) {
        const int i0 = min(i_base + (2 * k2) * 32, a.n_i - 1);
        const int i1 = min(i_base + (2 * k2 + 1) * 32, a.n_i - 1);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            ni[k2][c] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + c]), neg_canon(a.x_i[3 * (size_t)i1 + c]));
            ni[k2][3 + c] = pack2(-a.v_i[3 * (size_t)i0 + c], -a.v_i[3 * (size_t)i1 + c]);
        }
    }
    const u64 eps2_2 = pack2(a.eps2, a.eps2);
    // MODE_BLOOM: the filter of this warp's i-positions (nb_kernels.cuh; the WJ warps with the same wi share it)
    uint32_t* filt = reinterpret_cast<uint32_t*>(smem_raw + WJ * RING_BYTES + 2 * WJ * STAGES * 8) + wi * kBloomWords;
    if (MODE == MODE_BLOOM) {
        uint4* z = reinterpret_cast<uint4*>(smem_raw + WJ * RING_BYTES + 2 * WJ * STAGES * 8);
        for (int q = threadIdx.x; q < WI * kBloomWords / 4; q += 32 * WI * WJ) z[q] = make_uint4(0u, 0u, 0u, 0u);
        __syncthreads();
        if (wj == 0) {
#pragma unroll
            for (int k = 0; k < K; ++k) {
                const int i = min(i_base + k * 32, a.n_i - 1);
                bloom_set(filt, bloom_key(a.x_i[3 * (size_t)i + 0], a.x_i[3 * (size_t)i + 1], a.x_i[3 * (size_t)i + 2]));
            }
        }
    }
    __syncthreads();                                                   // barriers initialised, filters built

    if (producer) {
        const int pre = n_tiles < STAGES ? n_tiles : STAGES;
        for (int t = 0; t < pre; ++t) {
            const uint32_t bytes = (uint32_t)min(TJ, n_sub - t * TJ) * REC;
            mbar_expect_tx(full0 + 8 * t, bytes);
            tma_load_1d(ring + t * TJ * REC, src + (size_t)t * TJ * REC, bytes, full0 + 8 * t);
        }
    }

    double run[K][kHermiteAcc];
#pragma unroll
    for (int k = 0; k < K; ++k)
#pragma unroll
        for (int c = 0; c < kHermiteAcc; ++c) run[k][c] = 0.0;

    const int* coin = nullptr;
    int coin_cnt = 0, coin_pos = 0, coin_next = 0x7fffffff;
    if (MODE == MODE_LIST) {
        coin = a.coin_lists + (size_t)(blockIdx.x * WI + wi) * (1 + kCoinCap);
        coin_cnt = (*a.coin_flag != 0) ? -1 : coin[0];
        if (coin_cnt > 0) coin_next = coin[1];
    }

    for (int t = 0; t < n_tiles; ++t) {
        const int slot = t % STAGES;
        mbar_wait(full0 + 8 * slot, (uint32_t)(t / STAGES) & 1u);
        const int np = min(TJ, n_sub - t * TJ);
        const float4* sp = reinterpret_cast<const float4*>(rings + wj * RING_BYTES + slot * TJ * REC);
        for (int c = 0; c < np; c += SUB) {
            const int nc = min(SUB, np - c);
            u64 part[K / 2][kHermiteAcc];
            bool masked = true;
            if (MODE == MODE_LIST) {
                const int j0 = j_begin + t * TJ + c;
                const int seg_lo = j0 >> kCoinSegShift, seg_hi = (j0 + nc - 1) >> kCoinSegShift;
                while (coin_next < seg_lo) {
                    ++coin_pos;
                    coin_next = (coin_pos < coin_cnt) ? coin[1 + coin_pos] : 0x7fffffff;
                }
                masked = (coin_cnt < 0 || coin_next <= seg_hi);
            } else if (MODE == MODE_BLOOM) {
                bool hit = false;                                      // may a j of this block coincide with an i of this warp?
#pragma unroll
                for (int q = 0; q < SUB; q += 32) {                    // branch-free: 8 independent chains
                    const float4 J = sp[2 * (c + min(q + lane, nc - 1))];
                    hit |= bloom_test(filt, bloom_key(J.x, J.y, J.z));
                }
                masked = __any_sync(0xffffffffu, hit);
            }
            if (masked) hermite_sweep<K, true, PHI>(sp + 2 * c, nc, ni, eps2_2, part);
            else hermite_sweep<K, false, PHI>(sp + 2 * c, nc, ni, eps2_2, part);
#pragma unroll
            for (int k2 = 0; k2 < K / 2; ++k2)
#pragma unroll
                for (int q = 0; q < kHermiteAcc; ++q) {
                    float lo, hi;
                    unpack2(part[k2][q], lo, hi);
                    run[2 * k2][q] += (double)lo;
                    run[2 * k2 + 1][q] += (double)hi;
                }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
        if (producer) {
            const int tt = (WI > 1) ? t - 1 : t;
            if (tt >= 0 && tt + STAGES < n_tiles) {
                const int rs = tt % STAGES;
                mbar_wait(empty0 + 8 * rs, (uint32_t)(tt / STAGES) & 1u);
                const int tn = tt + STAGES;
                const uint32_t bytes = (uint32_t)min(TJ, n_sub - tn * TJ) * REC;
                mbar_expect_tx(full0 + 8 * rs, bytes);
                tma_load_1d(ring + rs * TJ * REC, src + (size_t)tn * TJ * REC, bytes, full0 + 8 * rs);
            }
        }
        __syncwarp();
    }

    if (WJ > 1) {
        __syncthreads();
        double* red = reinterpret_cast<double*>(smem_raw);             // [WJ][K][10][WI*32]
        const int tig = wi * 32 + lane;
#pragma unroll
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int c = 0; c < kHermiteAcc; ++c) red[((wj * K + k) * kHermiteAcc + c) * (WI * 32) + tig] = run[k][c];
        __syncthreads();
        if (!FUSED && wj != 0) return;
        if (wj == 0) {
#pragma unroll
            for (int k = 0; k < K; ++k)
#pragma unroll
                for (int c = 0; c < kHermiteAcc; ++c) {
                    double s = red[((0 * K + k) * kHermiteAcc + c) * (WI * 32) + tig];
#pragma unroll
                    for (int w = 1; w < WJ; ++w) s += red[((w * K + k) * kHermiteAcc + c) * (WI * 32) + tig];
                    run[k][c] = s;
                }
        }
    }

#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int i = i_base + k * 32;
        if (i >= a.n_i || wj != 0) continue;
        if (a.S == 1) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a.acc[3 * (size_t)i + c] = (float)run[k][c];
                a.jerk[3 * (size_t)i + c] = (float)(run[k][3 + c] - 3.0 * run[k][6 + c]);   // jk = jk1 - jk2
            }
            if (a.pot) a.pot[i] = -(float)run[k][9];
        } else {
            double* dst = a.partial + ((size_t)blockIdx.y * a.n_i + i) * kHermiteAcc;
#pragma unroll
            for (int c = 0; c < kHermiteAcc; c += 2) *reinterpret_cast<double2*>(dst + c) = make_double2(run[k][c], run[k][c + 1]);
        }
    }

    // second pass, fused (as in nb_force_kernel; MODE_EXACT instantiations only -- the small calls, where a launch
    // matters; the large-call kernels carry none of this): the CTA that finishes LAST among the S chunks of this i-tile sums the
    // S partials in the fixed order s = 0 .. S-1 -- the sum nb_hermite_reduce_kernel makes, bit for bit -- and writes
    // a, jerk and phi; the tile's ticket counter returns to zero for the next call.
    if (FUSED && a.S > 1 && a.tickets != nullptr) {
        __shared__ int s_last;
        __threadfence();                                               // partials visible device-wide before the ticket
        __syncthreads();
        if (threadIdx.x == 0) {
            const int ticket = atomicAdd(a.tickets + blockIdx.x, 1);
            s_last = (ticket == a.S - 1);
            if (s_last) a.tickets[blockIdx.x] = 0;
        }
        __syncthreads();
        if (!s_last) return;
        __threadfence();
        const int tile0 = blockIdx.x * (32 * K * WI);
        const int tile_n = min(32 * K * WI, a.n_i - tile0);
        for (int q = threadIdx.x; q < tile_n; q += 32 * WI * WJ) {
            const int i = tile0 + q;
            double s[kHermiteAcc];
            const double2* p2 = reinterpret_cast<const double2*>(a.partial + (size_t)i * kHermiteAcc);   // L2 reads
#pragma unroll
            for (int c = 0; c < kHermiteAcc; c += 2) { const double2 t = __ldcg(p2 + c / 2); s[c] = t.x; s[c + 1] = t.y; }
            for (int ch = 1; ch < a.S; ++ch) {
                p2 = reinterpret_cast<const double2*>(a.partial + ((size_t)ch * a.n_i + i) * kHermiteAcc);
#pragma unroll
                for (int c = 0; c < kHermiteAcc; c += 2) { const double2 t = __ldcg(p2 + c / 2); s[c] += t.x; s[c + 1] += t.y; }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a.acc[3 * (size_t)i + c] = (float)s[c];
                a.jerk[3 * (size_t)i + c] = (float)(s[3 + c] - 3.0 * s[6 + c]);
            }
            if (a.pot) a.pot[i] = -(float)s[9];
        }
    }
}

// second pass over the S chunk partials, fixed order
__global__ void __launch_bounds__(128) nb_hermite_reduce_kernel(const double* __restrict__ partial, int n_i, int S,
                                                                float* __restrict__ acc, float* __restrict__ jerk,
                                                                float* __restrict__ pot) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_i) return;
    double s[kHermiteAcc];
#pragma unroll
    for (int c = 0; c < kHermiteAcc; ++c) s[c] = partial[(size_t)i * kHermiteAcc + c];
    for (int q = 1; q < S; ++q) {
        const double* p = partial + ((size_t)q * n_i + i) * kHermiteAcc;
#pragma unroll
        for (int c = 0; c < kHermiteAcc; ++c) s[c] += p[c];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[3 * (size_t)i + c] = (float)s[c];
        jerk[3 * (size_t)i + c] = (float)(s[3 + c] - 3.0 * s[6 + c]);
    }
    if (pot) pot[i] = -(float)s[9];
}

// ---------------------------------------------------------------- shared-time-step Hermite integrator (O(N) kernels)
// predict:  xp = x + v dt + a dt^2/2 + j dt^3/6,   vp = v + a dt + j dt^2/2      (Horner form, FP32 FMAs)
// One thread per particle; it also writes the packed (x, y, z, m | vx, vy, vz, 0) records of the predicted state
// (what nb_pack_jv_kernel would write): a step of nb_hermite4 saves a launch and a pass over the particles.
__global__ void __launch_bounds__(256) nb_hermite_predict_pack_kernel(const float* __restrict__ x, const float* __restrict__ v,
                                                                      const float* __restrict__ a, const float* __restrict__ j,
                                                                      const float* __restrict__ m, float* __restrict__ xp,
                                                                      float* __restrict__ vp, float4* __restrict__ jp, int n, float dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float px[3], pv[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t k = 3 * (size_t)i + c;
        const float aa = a[k], jj = j[k], vv = v[k];
        px[c] = fmaf(fmaf(fmaf(jj, dt * (1.0f / 3.0f), aa), dt * 0.5f, vv), dt, x[k]);
        pv[c] = fmaf(fmaf(jj, dt * 0.5f, aa), dt, vv);
        xp[k] = px[c];
        vp[k] = pv[c];
    }
    jp[2 * (size_t)i + 0] = make_float4(px[0], px[1], px[2], m[i]);
    jp[2 * (size_t)i + 1] = make_float4(pv[0], pv[1], pv[2], 0.0f);
}
// correct:  v' = v + (a0 + a1) dt/2 + (j0 - j1) dt^2/12,   x' = x + (v + v') dt/2 + (a0 - a1) dt^2/12;   a0, j0 <- a1, j1
__global__ void __launch_bounds__(256) nb_hermite_correct_kernel(float* __restrict__ x, float* __restrict__ v,
                                                                 float* __restrict__ a0, float* __restrict__ j0,
                                                                 const float* __restrict__ a1, const float* __restrict__ j1,
                                                                 int n3, float dt) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n3) return;
    const float h = 0.5f * dt, h2 = dt * dt * (1.0f / 12.0f);
    const float a_old = a0[k], a_new = a1[k], j_old = j0[k], j_new = j1[k], v_old = v[k];
    const float v_new = fmaf(j_old - j_new, h2, fmaf(a_old + a_new, h, v_old));
    x[k] = fmaf(a_old - a_new, h2, fmaf(v_old + v_new, h, x[k]));
    v[k] = v_new;
    a0[k] = a_new;
    j0[k] = j_new;
}

// correct of step s and predict + pack of step s + 1 in one launch (one thread per particle; the same operations in the same
// order as the two kernels above, so the same bits): a step of nb_hermite4 is then two launches, which is what counts while
// the integration of a small system is launch-bound.
__global__ void __launch_bounds__(256) nb_hermite_correct_predict_pack_kernel(float* __restrict__ x, float* __restrict__ v,
                                                                              float* __restrict__ a0, float* __restrict__ j0,
                                                                              const float* __restrict__ a1, const float* __restrict__ j1,
                                                                              const float* __restrict__ m, float* __restrict__ xp,
                                                                              float* __restrict__ vp, float4* __restrict__ jp, int n, float dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float h = 0.5f * dt, h2 = dt * dt * (1.0f / 12.0f);
    float px[3], pv[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t k = 3 * (size_t)i + c;
        const float a_old = a0[k], a_new = a1[k], j_old = j0[k], j_new = j1[k], v_old = v[k];
        const float v_new = fmaf(j_old - j_new, h2, fmaf(a_old + a_new, h, v_old));
        const float x_new = fmaf(a_old - a_new, h2, fmaf(v_old + v_new, h, x[k]));
        x[k] = x_new;
        v[k] = v_new;
        a0[k] = a_new;
        j0[k] = j_new;
        px[c] = fmaf(fmaf(fmaf(j_new, dt * (1.0f / 3.0f), a_new), dt * 0.5f, v_new), dt, x_new);
        pv[c] = fmaf(fmaf(j_new, dt * 0.5f, a_new), dt, v_new);
        xp[k] = px[c];
        vp[k] = pv[c];
    }
    jp[2 * (size_t)i + 0] = make_float4(px[0], px[1], px[2], m[i]);
    jp[2 * (size_t)i + 1] = make_float4(pv[0], pv[1], pv[2], 0.0f);
}

// ---------------------------------------------------------------- block (individual) time steps: one block step, row f4
// Every particle holds (x, v, a, j) at its own time t[k] (FP64; the interval h = t_now - t[k] is rounded to FP32 once).
// predict everybody to t_now (same Horner form as the shared-step kernel, h per particle) and pack the j records:
// Predicted state of particle i at t_now (shared by both halves of the kernel below, so the due particles' i-records
// are bitwise the j-records of the same particles: the coincidence test sees each particle's own record).
__device__ __forceinline__ void nb_block_predict(const float* __restrict__ x, const float* __restrict__ v,
                                                 const float* __restrict__ a, const float* __restrict__ j,
                                                 const double* __restrict__ t, double t_now, int i, float px[3], float pv[3]) {
    const float dt = (float)(t_now - t[i]);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t k = 3 * (size_t)i + c;
        const float aa = a[k], jj = j[k], vv = v[k];
        px[c] = fmaf(fmaf(fmaf(jj, dt * (1.0f / 3.0f), aa), dt * 0.5f, vv), dt, x[k]);
        pv[c] = fmaf(fmaf(jj, dt * 0.5f, aa), dt, vv);
    }
}
// CTAs [0, j_blocks): everybody's packed j record (and xp, vp); CTAs [j_blocks, ...): the i-set = predicted state of the
// due particles in the order of active[] (one launch instead of a prediction and a gather)
__global__ void __launch_bounds__(256) nb_block_predict_pack_kernel(const float* __restrict__ x, const float* __restrict__ v,
                                                                    const float* __restrict__ a, const float* __restrict__ j,
                                                                    const float* __restrict__ m, const double* __restrict__ t,
                                                                    double t_now, float* __restrict__ xp, float* __restrict__ vp,
                                                                    float4* __restrict__ jp, int n, int j_blocks,
                                                                    const int* __restrict__ active, int n_act,
                                                                    float* __restrict__ xi, float* __restrict__ vi) {
    float px[3], pv[3];
    if ((int)blockIdx.x < j_blocks) {
        const int i = blockIdx.x * blockDim.x + threadIdx.x;
        if (i >= n) return;
        nb_block_predict(x, v, a, j, t, t_now, i, px, pv);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xp[3 * (size_t)i + c] = px[c];
            vp[3 * (size_t)i + c] = pv[c];
        }
        jp[2 * (size_t)i + 0] = make_float4(px[0], px[1], px[2], m[i]);
        jp[2 * (size_t)i + 1] = make_float4(pv[0], pv[1], pv[2], 0.0f);
    } else {
        const int q = ((int)blockIdx.x - j_blocks) * blockDim.x + threadIdx.x;
        if (q >= n_act) return;
        nb_block_predict(x, v, a, j, t, t_now, active[q], px, pv);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xi[3 * (size_t)q + c] = px[c];
            vi[3 * (size_t)q + c] = pv[c];
        }
    }
}
// correct the active particles over their own interval and advance their clocks; nobody else is written
__global__ void __launch_bounds__(256) nb_block_correct_kernel(float* __restrict__ x, float* __restrict__ v,
                                                               float* __restrict__ a0, float* __restrict__ j0,
                                                               double* __restrict__ t, const int* __restrict__ active,
                                                               const float* __restrict__ a1, const float* __restrict__ j1,
                                                               double t_now, int n_act) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_act) return;
    const int i = active[q];
    const float dt = (float)(t_now - t[i]);
    const float h = 0.5f * dt, h2 = dt * dt * (1.0f / 12.0f);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t k = 3 * (size_t)i + c, e = 3 * (size_t)q + c;
        const float a_old = a0[k], a_new = a1[e], j_old = j0[k], j_new = j1[e], v_old = v[k];
        const float v_new = fmaf(j_old - j_new, h2, fmaf(a_old + a_new, h, v_old));
        x[k] = fmaf(a_old - a_new, h2, fmaf(v_old + v_new, h, x[k]));
        v[k] = v_new;
        a0[k] = a_new;
        j0[k] = j_new;
    }
    t[i] = t_now;
}

// ---------------------------------------------------------------- block-step scheduler: who is due next (index work, exact)
// t_next = min_k (t[k] + dt[k]);  active = ascending { k : t[k] + dt[k] == t_next }.  One FP64 add per particle, the same
// on both passes, so the equality is exact.  A CTA covers kSchedTile consecutive particles, a thread kSchedItems of them.
// A due time that is not finite (a particle parked with dt = +inf, a NaN clock, -inf) is never the minimum and never due.
constexpr int kSchedThreads = 256, kSchedItems = 4, kSchedTile = kSchedThreads * kSchedItems;
__device__ __forceinline__ bool nb_sched_finite(double due) { return fabs(due) <= 1.7976931348623157e308; }   // false for NaN

__global__ void __launch_bounds__(kSchedThreads) nb_sched_min_kernel(const double* __restrict__ t, const double* __restrict__ dt,
                                                                    int n, double* __restrict__ block_min) {
    __shared__ double warp_min[kSchedThreads / 32];
    const size_t base = (size_t)blockIdx.x * kSchedTile + (size_t)threadIdx.x * kSchedItems;
    double lo = CUDART_INF;
#pragma unroll
    for (int e = 0; e < kSchedItems; ++e)
        if (base + e < (size_t)n) {
            const double due_k = __dadd_rn(t[base + e], dt[base + e]);
            if (nb_sched_finite(due_k)) lo = fmin(lo, due_k);
        }
    for (int o = 16; o > 0; o >>= 1) lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    if ((threadIdx.x & 31) == 0) warp_min[threadIdx.x >> 5] = lo;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kSchedThreads / 32; ++w) lo = fmin(lo, warp_min[w]);
        block_min[blockIdx.x] = lo;
    }
}
// one CTA: the minimum of the CTA minima (+inf when there is no particle)
__global__ void __launch_bounds__(1024) nb_sched_final_min_kernel(const double* __restrict__ block_min, int n_blocks,
                                                                  double* __restrict__ t_next) {
    __shared__ double warp_min[32];
    double lo = CUDART_INF;
    for (int b = threadIdx.x; b < n_blocks; b += 1024) lo = fmin(lo, block_min[b]);
    for (int o = 16; o > 0; o >>= 1) lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    if ((threadIdx.x & 31) == 0) warp_min[threadIdx.x >> 5] = lo;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 32; ++w) lo = fmin(lo, warp_min[w]);
        *t_next = lo;
    }
}
// how many of a CTA's particles are due
__global__ void __launch_bounds__(kSchedThreads) nb_sched_count_kernel(const double* __restrict__ t, const double* __restrict__ dt,
                                                                      int n, const double* __restrict__ t_next,
                                                                      int* __restrict__ counts) {
    __shared__ int total;
    if (threadIdx.x == 0) total = 0;
    __syncthreads();
    const double due = *t_next;
    const size_t base = (size_t)blockIdx.x * kSchedTile + (size_t)threadIdx.x * kSchedItems;
    int c = 0;
#pragma unroll
    for (int e = 0; e < kSchedItems; ++e)
        if (base + e < (size_t)n) c += (__dadd_rn(t[base + e], dt[base + e]) == due && nb_sched_finite(due));
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(&total, c);          // integer sum: the order does not matter
    __syncthreads();
    if (threadIdx.x == 0) counts[blockIdx.x] = total;
}
// one CTA: exclusive scan of the CTA counts in place, the grand total to n_act
__global__ void __launch_bounds__(1024) nb_sched_scan_kernel(int* __restrict__ counts, int n_blocks, int* __restrict__ n_act) {
    __shared__ int buf[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int c0 = 0; c0 < n_blocks; c0 += 1024) {
        const int b = c0 + threadIdx.x;
        const int mine = b < n_blocks ? counts[b] : 0;
        buf[threadIdx.x] = mine;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {                          // Hillis-Steele inclusive scan
            const int add = threadIdx.x >= o ? buf[threadIdx.x - o] : 0;
            __syncthreads();
            buf[threadIdx.x] += add;
            __syncthreads();
        }
        const int before = carry;
        if (b < n_blocks) counts[b] = before + buf[threadIdx.x] - mine;
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + buf[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_act = carry;
}
// the due particles' indices, ascending: CTA offset + position inside the CTA
__global__ void __launch_bounds__(kSchedThreads) nb_sched_scatter_kernel(const double* __restrict__ t, const double* __restrict__ dt,
                                                                        int n, const double* __restrict__ t_next,
                                                                        const int* __restrict__ offsets, int* __restrict__ active) {
    __shared__ int warp_sum[kSchedThreads / 32];
    const double due = *t_next;
    const size_t base = (size_t)blockIdx.x * kSchedTile + (size_t)threadIdx.x * kSchedItems;
    bool flag[kSchedItems];
    int c = 0;
#pragma unroll
    for (int e = 0; e < kSchedItems; ++e) {
        flag[e] = base + e < (size_t)n && __dadd_rn(t[base + e], dt[base + e]) == due && nb_sched_finite(due);
        c += flag[e];
    }
    int incl = c;                                                      // inclusive scan over the warp
    for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, incl, o);
        if ((threadIdx.x & 31) >= o) incl += up;
    }
    if ((threadIdx.x & 31) == 31) warp_sum[threadIdx.x >> 5] = incl;
    __syncthreads();
    int pos = offsets[blockIdx.x] + incl - c;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) pos += warp_sum[w];
#pragma unroll
    for (int e = 0; e < kSchedItems; ++e)
        if (flag[e]) active[pos++] = (int)(base + e);
}

// ---------------------------------------------------------------- block-step size: the Aarseth criterion, FP32, fixed order
// dt = sqrt(eta (|a1||a2'| + |j1|^2) / (|j1||a3| + |a2'|^2)) from the Hermite interpolant of (a0, j0) -> (a1, j1) over h.
// The value feeds an integer decision (the block level), so every operation is one explicitly rounded FP32 operation
// (no FMA contraction, IEEE division and square root), in the order the header states.
__device__ __forceinline__ float nb_norm2_rn(const float z[3]) {
    return __fadd_rn(__fadd_rn(__fmul_rn(z[0], z[0]), __fmul_rn(z[1], z[1])), __fmul_rn(z[2], z[2]));
}
__global__ void __launch_bounds__(256) nb_block_step_size_kernel(const float* __restrict__ a0, const float* __restrict__ j0,
                                                                 const float* __restrict__ a1, const float* __restrict__ j1,
                                                                 const float* __restrict__ h, float eta, float* __restrict__ dt_out,
                                                                 int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float hh = h[i];
    const float h2 = __fmul_rn(hh, hh), h3 = __fmul_rn(h2, hh), h6 = __fmul_rn(6.0f, hh);
    float va1[3], vj1[3], va2[3], va3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t k = 3 * (size_t)i + c;
        const float p0 = a0[k], q0 = j0[k], p1 = a1[k], q1 = j1[k];
        const float da = __fsub_rn(p0, p1);
        const float s1 = __fadd_rn(__fmul_rn(4.0f, q0), __fmul_rn(2.0f, q1));
        const float a2 = __fdiv_rn(-__fadd_rn(__fmul_rn(6.0f, da), __fmul_rn(hh, s1)), h2);
        const float s2 = __fadd_rn(q0, q1);
        const float a3 = __fdiv_rn(__fadd_rn(__fmul_rn(12.0f, da), __fmul_rn(h6, s2)), h3);
        va1[c] = p1;
        vj1[c] = q1;
        va3[c] = a3;
        va2[c] = __fadd_rn(a2, __fmul_rn(hh, a3));
    }
    const float a1sq = nb_norm2_rn(va1), j1sq = nb_norm2_rn(vj1), a2sq = nb_norm2_rn(va2), a3sq = nb_norm2_rn(va3);
    const float top = __fadd_rn(__fmul_rn(__fsqrt_rn(a1sq), __fsqrt_rn(a2sq)), j1sq);
    const float bot = __fadd_rn(__fmul_rn(__fsqrt_rn(j1sq), __fsqrt_rn(a3sq)), a2sq);
    dt_out[i] = __fsqrt_rn(__fmul_rn(eta, __fdiv_rn(top, bot)));
}

}  // namespace nb
