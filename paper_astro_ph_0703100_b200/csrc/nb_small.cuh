// nb_small.cuh -- the force kernel for SMALL i-sets (row a7 of SURVEY.md section 8: the j-split mode; BASELINE.json
// configs[0] and configs[2]; section 4.4: calls with few i-particles are where a tree code spends
// its time).
//
// Why a second kernel.  nb_force_kernel packs TWO i-particles into every f32x2 instruction; with few i-particles a
// thread then holds one packed pair (K = 2), the loop has one dependent chain, and every j costs a shared-memory load
// for 13 packed instructions: C2 (512 x 65536) ran at 35 % of the FP32 roofline, C0 (2048 x 2048) at 12 %
// (profiles/r02_small_calls.md).  Here the roles inside a packed instruction flip:
//
//   * PACKED OVER j: the two halves of an f32x2 register hold two CONSECUTIVE j-particles, the i-particle is the
//     32-bit broadcast operand (SASS: FADD2 R, R.F32x2, R.F32).  One thread with ONE i-particle fills both halves;
//     its two LDS.128 per j-pair feed 13 packed instructions for each of its KI i-particles.
//   * shared memory holds the j-particles already interleaved as pairs, (x0,x1,y0,y1) (z0,z1,m0,m1), written there by
//     the CTA itself from x_j / m_j (rows a1 + a2 in one step: no pack launch, no TMA round trip -- a CTA's share of
//     the j-range is a few hundred particles);
//   * the lanes of a warp may be split LI x LJ: LI i-particles x LJ j-slots, so that 16 or 8 i-particles per warp still
//     use 32 lanes (C0: 2048 i-particles must cover 148 SMs x 8 warps);
//   * the j-range is split over LJ lanes x WJ warps x S CTAs; the partial sums are combined in a FIXED order at every
//     level: shuffles (LJ), shared memory (WJ), DISTRIBUTED shared memory inside a thread-block cluster of CS CTAs
//     (each CTA of the cluster sums a slice of the i-tile over the cluster's CTAs), and -- only when S > CS -- FP64
//     partials in global memory, summed by the last-arriving CTA of every (i-tile, slice).  No floating-point atomics:
//     bitwise reproducible, invariant under permutation of the i-set.
//
// Arithmetic per pair is that of pair_body() in nb_kernels.cuh (Fig. A.3; phi as in Fig. A.4,
// PAPER.md:509-516, 552): 13 FP32-pipe instructions + 1 MUFU per pair; Eq. (2): FP32 partial sums over at
// most 128 consecutive j of a slot, FP64 running totals.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "../../include/nb_packed.cuh"

namespace nb {

struct SmallArgs {
    const float* x_i;      // [n_i][3]
    const float* xj_raw;   // [n_j][3]   (nullptr when jp is given)
    const float* mj_raw;   // [n_j]
    const float4* jp;      // packed (x, y, z, m) records: nb_force_packed
    float* acc;            // [n_i][3]
    float* pot;            // [n_i] or nullptr
    double4* partial;      // [n_i][S / CS] when S > CS
    int* tickets;          // [tiles_i * CS] zero between calls, when S > CS
    int n_i;
    int n_j;
    int S;                 // j-chunks across CTAs (grid.y), a multiple of CS
    int flag_offset;       // SMALL_FLAG: byte offset of the tile's Bloom filter + the slot bitmaps in dynamic shared memory
#ifdef NB_SMALL_STAMPS
    long long* stamps;     // working builds only: [n_ctas][16] %globaltimer and clock64 stamps of the kernel's phases
#endif
    float eps2;
};

constexpr int kSmallThreadsMax = 512;
constexpr int kSmallRoundJ = 4096;     // j-particles staged in shared memory at a time (64 KB + padding)
constexpr int kSmallLoadBatch = 4;     // j-pairs a thread loads before it stores them to shared memory
constexpr int kSmallBlockPairs = 64;   // Eq. (2): FP32 partial sums run over at most 64 j-pairs = 128 j of a slot (= one 64-bit
                                       // word of the SMALL_FLAG bitmap of marked pairs)

// ---------------------------------------------------------------- thread-block cluster helpers
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_map_shared(uint32_t smem_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ double2 cluster_ld_double2(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}

// ---------------------------------------------------------------- one i-particle x two j-particles
// xj2 = (x_j0, x_j1) etc.; nxi = (-x_i, -x_i) (ptxas folds the duplicate into the .F32 broadcast operand form).
template <int MASK, bool PHI>
__device__ __forceinline__ void pair_body_j2(u64 xj2, u64 yj2, u64 zj2, u64 mj2, u64 nxi, u64 nyi, u64 nzi, u64 eps2_2,
                                             u64& ax, u64& ay, u64& az, u64& ph) {
    const u64 dx = add2(xj2, nxi);                   // dx = xj - xi
    const u64 dy = add2(yj2, nyi);
    const u64 dz = add2(zj2, nzi);
    u64 r2 = fma2(dx, dx, eps2_2);                   // r2 = dx2+dy2+dz2+eps2 PAPER.md:464
    r2 = fma2(dy, dy, r2);
    r2 = fma2(dz, dz, r2);
    float r2a, r2b;
    unpack2(r2, r2a, r2b);
    if (MASK == MASK_EXACT) {                        // reading R1: all three differences exactly zero -> the pair adds nothing
        const float inf = __int_as_float(0x7f800000);
        float dxa, dxb, dya, dyb, dza, dzb;
        unpack2(dx, dxa, dxb); unpack2(dy, dya, dyb); unpack2(dz, dza, dzb);
        const uint32_t ta = __float_as_uint(dxa) | __float_as_uint(dya) | __float_as_uint(dza);
        const uint32_t tb = __float_as_uint(dxb) | __float_as_uint(dyb) | __float_as_uint(dzb);
        r2a = (ta == 0u) ? inf : r2a;                // rsqrt(+inf) = +0
        r2b = (tb == 0u) ? inf : r2b;
    }
    const u64 u = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));   // r1i = 1/sqrt(r2)
    const u64 u2 = mul2(u, u);                       // r2i
    const u64 mu = mul2(mj2, u);                     // pot = mj * r1i
    const u64 mu3 = mul2(mu, u2);                    // mr3i
    ax = fma2(mu3, dx, ax);                          // OUTPUT[0..2] += mr3i*d PAPER.md:469-471
    ay = fma2(mu3, dy, ay);
    az = fma2(mu3, dz, az);
    if (PHI) ph = add2(ph, mu);                      // OUTPUT[6] -= pot (sign at the end) PAPER.md:552
}


// Shared-memory stride of a j-slot, in pairs: odd, so that the LJ lanes groups of a warp, which read the same pair
// index of LJ different slots, fall on different banks (32 B per pair: odd multiples of 32 B are distinct mod 128 B).
__host__ __device__ inline int small_slot_len(int round_j, int Q) {   // j-particles per slot, even
    const int l = (round_j + Q - 1) / Q;
    return (l + 1) & ~1;
}
__host__ __device__ inline int small_pair_stride(int slot_len) { return (slot_len / 2) | 1; }

// ---------------------------------------------------------------- the kernel
// CTA = 8 warps = WI (along i) x WJ (along j); lanes = LI (along i) x LJ (along j); KI i-particles per thread.
// i-tile of a CTA = WI * KI * LI particles; the CTA's j-chunk (blockIdx.y of S) is cut into Q = WJ * LJ slots.
// NW = warps per CTA (8 or 16); CS = 1: no cluster; CS = 8: launched in clusters of 2, 4 or 8 CTAs along grid.y.
//
// Coincident pairs (reading R1), MODE:
//   SMALL_EXACT  every pair masked (LOP3 + FSEL per pair on the ALU pipe): the loop reaches 62-70 % of the FP32 roofline
//                where the unmasked loop reaches 69-85 % (profiles/r02_microloops.md);
//   SMALL_NONE   no mask: valid without phi for eps2 >= 2^-40 (an unmasked coincident pair adds m u^3 (+-0) to a);
//   SMALL_FLAG   (LJ = 1, eps2 >= 2^-40) the j-PAIRS that may hold a coincident particle are marked while they are staged:
//                the CTA builds a Bloom filter of its tile's i-positions (nb_packed.cuh; no false negatives), every staged
//                j is tested once, and a hit sets the pair's bit in a per-slot bitmap.  All lanes of a warp sweep the same
//                pair, so the loop branches warp-uniformly: runs of unmarked pairs go through the unmasked body, a marked
//                pair through the masked one.  Same pairs, same order, and the two bodies give the same bits for a pair
//                that is not coincident: the result is the always-masked one bit for bit (a false positive only costs
//                the mask), whatever the tile holds -- invariant under permutation of the i-set.
// Two cheaper ways to honour the rule were built and measured on C2 and dropped: a per-warp Bloom
// filter tested per Eq. (2) block (the CTA lasts as long as its slowest warp, and with one or two blocks per warp the
// masked ones set the pace: 26.3 against 25.7 us), and a hash join of the staged j-particles against the CTA's i-tile
// with the coincident ones swept separately (the probe made staging 4x slower, and a sum order that depends on which
// particles share a tile is not invariant under permutation of the i-set).
enum { SMALL_EXACT = 0, SMALL_FLAG = 1, SMALL_NONE = 2 };
__host__ __device__ inline int small_flag_words(int pstride) { return (pstride + 63) >> 6; }   // 64-bit words per slot bitmap

template <int NW, int KI, int LJ, int WJ, int MODE, bool PHI, int CS>
__global__ void __launch_bounds__(32 * NW) nb_small_kernel(const SmallArgs a) {
    constexpr int WI = NW / WJ, LI = 32 / LJ, Q = WJ * LJ, TILE_I = WI * KI * LI, kSmallThreads = 32 * NW;
    static_assert(WI * WJ == NW && LI * LJ == 32, "NW warps of 32 lanes");
    static_assert(MODE == SMALL_EXACT || MODE == SMALL_FLAG || MODE == SMALL_NONE, "masked everywhere, marked pairs only, or no mask");
    static_assert(MODE != SMALL_FLAG || LJ == 1, "the marked-pair branch must be warp-uniform");
    static_assert(TILE_I % CS == 0, "every CTA of a cluster sums a whole slice of the i-tile");
    extern __shared__ __align__(128) unsigned char smem_raw[];
#ifdef NB_SMALL_STAMPS
#define NB_STAMP(k) do { if (a.stamps && threadIdx.x == 0) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); \
        a.stamps[(size_t)(blockIdx.y * gridDim.x + blockIdx.x) * 16 + (k)] = t_; \
        a.stamps[(size_t)(blockIdx.y * gridDim.x + blockIdx.x) * 16 + 8 + (k)] = clock64(); } } while (0)
#else
#define NB_STAMP(k) do { } while (0)
#endif
    // Programmatic dependent launch (nb_small_launch.cu sets the attribute): this grid may be scheduled while the previous
    // kernel of the stream is still draining; nothing of its output -- nor the ticket counters -- is touched before this wait.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    NB_STAMP(0);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wi = warp % WI, wj = warp / WI;
    const int li = lane % LI, lj = lane / LI;
    const int q = wj * LJ + lj;                                        // this thread's j-slot
    const int tile0 = blockIdx.x * TILE_I;

    // a3: i-particles of this thread (clamped loads; stores are guarded); -x_i with zeros canonicalised (nb_packed.cuh)
    u64 nxi[KI], nyi[KI], nzi[KI];
#pragma unroll
    for (int k = 0; k < KI; ++k) {
        const int i = min(tile0 + (wi * KI + k) * LI + li, a.n_i - 1);
        const float x = neg_canon(a.x_i[3 * (size_t)i + 0]), y = neg_canon(a.x_i[3 * (size_t)i + 1]),
                    z = neg_canon(a.x_i[3 * (size_t)i + 2]);
        nxi[k] = pack2(x, x); nyi[k] = pack2(y, y); nzi[k] = pack2(z, z);
    }
    const u64 eps2_2 = pack2(a.eps2, a.eps2);

    double run[KI][4];                                                 // running totals (outer level of Eq. (2))
#pragma unroll
    for (int k = 0; k < KI; ++k) { run[k][0] = run[k][1] = run[k][2] = run[k][3] = 0.0; }

    // the CTA's j-chunk (even boundaries, so that a j-pair never straddles two CTAs), staged in rounds of at most
    // kSmallRoundJ particles
    const int c_lo = (blockIdx.y == 0) ? 0 : ((int)((long long)a.n_j * blockIdx.y / a.S) & ~1);
    const int c_hi = ((int)blockIdx.y + 1 == a.S) ? a.n_j : ((int)((long long)a.n_j * (blockIdx.y + 1) / a.S) & ~1);
    const int chunk_max = (a.n_j + a.S - 1) / a.S + 2;
    const int round_max = min(kSmallRoundJ, chunk_max);
    const int slot_len = small_slot_len(round_max, Q);
    const int pstride = small_pair_stride(slot_len);
    float4* sj = reinterpret_cast<float4*>(smem_raw);                  // [Q][pstride][2]: (x0 x1 y0 y1) (z0 z1 m0 m1)
    // 8-byte loads of two consecutive particles need 8-byte aligned arrays (c_lo and every pair index are even)
    const bool wide = a.jp == nullptr && ((reinterpret_cast<uintptr_t>(a.xj_raw) | reinterpret_cast<uintptr_t>(a.mj_raw)) & 7u) == 0;

    // SMALL_FLAG: Bloom filter of the tile's i-positions, then one bitmap of marked pairs per j-slot
    uint32_t* filt = reinterpret_cast<uint32_t*>(smem_raw + a.flag_offset);
    unsigned long long* sbits = reinterpret_cast<unsigned long long*>(filt + kBloomWords);
    const int sw = small_flag_words(pstride);
    if (MODE == SMALL_FLAG) {
        for (int w = threadIdx.x; w < kBloomWords; w += kSmallThreads) filt[w] = 0u;
        for (int w = threadIdx.x; w < Q * sw; w += kSmallThreads) sbits[w] = 0ull;
        __syncthreads();
        for (int il = threadIdx.x; il < TILE_I; il += kSmallThreads) {
            const int i = tile0 + il;
            if (i < a.n_i) bloom_set(filt, bloom_key(a.x_i[3 * (size_t)i + 0], a.x_i[3 * (size_t)i + 1], a.x_i[3 * (size_t)i + 2]));
        }
        __syncthreads();
    }

    // a1 + a2: the CTA packs a round into the interleaved pair layout (Fig. A.1 packing loop).  One thread
    // per j-pair; the loads of kSmallLoadBatch pairs are in flight together (one memory latency per batch).
    auto stage_round = [&](int r_lo, int nr) {
        const int n_pairs_round = (nr + 1) >> 1;
        for (int p0 = threadIdx.x; p0 < n_pairs_round; p0 += kSmallThreads * kSmallLoadBatch) {
            float4 A[kSmallLoadBatch], B[kSmallLoadBatch];
#pragma unroll
            for (int u = 0; u < kSmallLoadBatch; ++u) {
                const int pp = p0 + u * kSmallThreads;
                if (pp >= n_pairs_round) break;
                const size_t j = (size_t)r_lo + 2 * (size_t)pp;
                const bool two = 2 * pp + 1 < nr;                      // false: the round's last pair holds one particle
                if (a.jp) {
                    const float4 J0 = a.jp[j], J1 = two ? a.jp[j + 1] : make_float4(J0.x, J0.y, J0.z, 0.0f);
                    A[u] = make_float4(J0.x, J1.x, J0.y, J1.y); B[u] = make_float4(J0.z, J1.z, J0.w, J1.w);
                } else if (wide && two) {
                    const float2* xp = reinterpret_cast<const float2*>(a.xj_raw + 3 * j);   // x0 y0 | z0 x1 | y1 z1
                    const float2 v0 = xp[0], v1 = xp[1], v2 = xp[2];
                    const float2 mm = *reinterpret_cast<const float2*>(a.mj_raw + j);
                    A[u] = make_float4(v0.x, v1.y, v0.y, v2.x); B[u] = make_float4(v1.x, v2.y, mm.x, mm.y);
                } else {
                    const float x0 = a.xj_raw[3 * j + 0], y0 = a.xj_raw[3 * j + 1], z0 = a.xj_raw[3 * j + 2], m0 = a.mj_raw[j];
                    // an odd count: the second half is a copy with zero mass (adds nothing)
                    const float x1 = two ? a.xj_raw[3 * j + 3] : x0, y1 = two ? a.xj_raw[3 * j + 4] : y0,
                                z1 = two ? a.xj_raw[3 * j + 5] : z0, m1 = two ? a.mj_raw[j + 1] : 0.0f;
                    A[u] = make_float4(x0, x1, y0, y1); B[u] = make_float4(z0, z1, m0, m1);
                }
            }
#pragma unroll
            for (int u = 0; u < kSmallLoadBatch; ++u) {
                const int pp = p0 + u * kSmallThreads;
                if (pp >= n_pairs_round) break;
                const int jj = 2 * pp, sq = jj / slot_len, pos = jj - sq * slot_len;
                float4* d = sj + ((size_t)sq * pstride + (pos >> 1)) * 2;
                d[0] = A[u]; d[1] = B[u];
                if (MODE == SMALL_FLAG) {                              // may one of the two coincide with an i-particle of the tile?
                    const bool hit = bloom_test(filt, bloom_key(A[u].x, A[u].z, B[u].x)) | bloom_test(filt, bloom_key(A[u].y, A[u].w, B[u].y));
                    if (hit) atomicOr(&sbits[sq * sw + (pos >> 7)], 1ull << ((pos >> 1) & 63));
                }
            }
        }
    };

    for (int r_lo = c_lo; r_lo < c_hi; r_lo += kSmallRoundJ) {
        const int nr = min(kSmallRoundJ, c_hi - r_lo);
        if (r_lo != c_lo) {
            __syncthreads();                                           // the previous round has been consumed
            if (MODE == SMALL_FLAG) {
                for (int w = threadIdx.x; w < Q * sw; w += kSmallThreads) sbits[w] = 0ull;
                __syncthreads();
            }
        }
        stage_round(r_lo, nr);
        __syncthreads();
        NB_STAMP(1);

        const int len_q = max(0, min(slot_len, nr - q * slot_len));
        const int npairs = (len_q + 1) >> 1;
        const float4* sp = sj + (size_t)q * pstride * 2;
        // Eq. (2) blocks: FP32 partial sums over at most kSmallBlockPairs pairs, then added to the running totals
        for (int b = 0; b < npairs; b += kSmallBlockPairs) {
            const int nb_ = min(kSmallBlockPairs, npairs - b);
            u64 pax[KI], pay[KI], paz[KI], pph[KI];
#pragma unroll
            for (int k = 0; k < KI; ++k) { pax[k] = 0ull; pay[k] = 0ull; paz[k] = 0ull; pph[k] = 0ull; }
            auto sweep = [&](auto mask_tag, int p_lo, int p_hi) {
                constexpr int MASK = decltype(mask_tag)::value;
#pragma unroll(KI == 2 ? 4 : 8)
                for (int p = p_lo; p < p_hi; ++p) {
                    const float4 A = sp[2 * (b + p)], B = sp[2 * (b + p) + 1];   // two LDS.128: (x0 x1 y0 y1) (z0 z1 m0 m1)
                    const u64 xj2 = pack2(A.x, A.y), yj2 = pack2(A.z, A.w), zj2 = pack2(B.x, B.y), mj2 = pack2(B.z, B.w);
#pragma unroll
                    for (int k = 0; k < KI; ++k)
                        pair_body_j2<MASK, PHI>(xj2, yj2, zj2, mj2, nxi[k], nyi[k], nzi[k], eps2_2, pax[k], pay[k], paz[k], pph[k]);
                }
            };
            if (MODE == SMALL_FLAG) {
                // groups of U pairs (the unroll width, so every group keeps U independent chains in flight): a group with a
                // marked pair runs masked, the others unmasked -- whatever the density of marks, never slower than SMALL_EXACT
                // in the loop (runs between single marks fell into the unrolled loops' remainders: 60 % slower at 1 mark in 32)
                constexpr int U = (KI == 2) ? 4 : 8;
                const unsigned long long word = sbits[q * sw + (b >> 6)];      // warp-uniform (LJ = 1): kSmallBlockPairs = 64 pairs per word
                int p = 0;
                for (; p + U <= nb_; p += U) {
                    if ((word >> p) & ((1ull << U) - 1ull)) sweep(std::integral_constant<int, MASK_EXACT>{}, p, p + U);
                    else sweep(std::integral_constant<int, MASK_NONE>{}, p, p + U);
                }
                if (p < nb_) sweep(std::integral_constant<int, MASK_EXACT>{}, p, nb_);
            } else if (MODE == SMALL_EXACT) {
                sweep(std::integral_constant<int, MASK_EXACT>{}, 0, nb_);
            } else {
                sweep(std::integral_constant<int, MASK_NONE>{}, 0, nb_);
            }
#pragma unroll
            for (int k = 0; k < KI; ++k) {                             // a5: even-j half first, then odd-j half
                float lo, hi;
                unpack2(pax[k], lo, hi); run[k][0] += (double)lo; run[k][0] += (double)hi;
                unpack2(pay[k], lo, hi); run[k][1] += (double)lo; run[k][1] += (double)hi;
                unpack2(paz[k], lo, hi); run[k][2] += (double)lo; run[k][2] += (double)hi;
                if (PHI) { unpack2(pph[k], lo, hi); run[k][3] += (double)lo; run[k][3] += (double)hi; }
            }
        }
    }

    NB_STAMP(2);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");    // the pair loop is done: the next launch may start scheduling
    // a7, level 1: the LJ lanes that hold the same i-particle, in the order lj = 0 .. LJ-1 (every lane forms the same sum)
    if (LJ > 1) {
#pragma unroll
        for (int k = 0; k < KI; ++k)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const double v = run[k][c];
                double s = __shfl_sync(0xffffffffu, v, li);
#pragma unroll
                for (int t = 1; t < LJ; ++t) s += __shfl_sync(0xffffffffu, v, li + t * LI);
                run[k][c] = s;
            }
    }

    // a7, level 2: the WJ warps that hold the same i-particles, through shared memory, in the order wj = 0 .. WJ-1
    __syncthreads();                                                   // the staged j-particles are dead: reuse the memory
    double4* red = reinterpret_cast<double4*>(smem_raw);               // [WJ][TILE_I]   (WJ > 1 only)
    double4* tile_sum = red + (WJ > 1 ? WJ * TILE_I : 0);              // [TILE_I]
    if (lj == 0) {
#pragma unroll
        for (int k = 0; k < KI; ++k) {
            const int il = (wi * KI + k) * LI + li;
            (WJ > 1 ? red[wj * TILE_I + il] : tile_sum[il]) = make_double4(run[k][0], run[k][1], run[k][2], run[k][3]);
        }
    }
    if (WJ > 1) {
        __syncthreads();
        for (int il = threadIdx.x; il < TILE_I; il += kSmallThreads) {
            double4 s = red[il];
#pragma unroll
            for (int w = 1; w < WJ; ++w) {
                const double4 v = red[w * TILE_I + il];
                s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
            }
            tile_sum[il] = s;
        }
    }

    // a7, level 3: the CS CTAs of the cluster (consecutive j-chunks of the same i-tile), through distributed shared
    // memory: CTA r of the cluster sums slice r of the tile over the cluster's CTAs in rank order.
    // (the instantiation CS = kSmallClusterMax serves every launched cluster size cs = 2, 4, 8: cs is read from the
    // hardware, the loads of absent ranks are predicated off)
    const int cs = (CS > 1) ? (int)cluster_nctarank() : 1;
    const int SLICE = TILE_I / cs;
    const uint32_t rank = (CS > 1) ? cluster_ctarank() : 0u;
    if (CS > 1) cluster_sync_all(); else __syncthreads();
    const int n_groups = a.S / cs;                                     // cluster partials per i-tile
    const int group = blockIdx.y / cs;
    for (int t = threadIdx.x; t < SLICE; t += kSmallThreads) {
        const int il = (int)rank * SLICE + t;
        double4 s;
        if (CS > 1) {
            const uint32_t local = smem_u32(tile_sum + il);
            double2 lo[CS], hi[CS];
#pragma unroll
            for (int c = 0; c < CS; ++c) {                             // all loads in flight, then the adds in rank order
                lo[c] = hi[c] = make_double2(0.0, 0.0);
                if (c < cs) { lo[c] = cluster_ld_double2(cluster_map_shared(local, c)); hi[c] = cluster_ld_double2(cluster_map_shared(local + 16, c)); }
            }
            s = make_double4(lo[0].x, lo[0].y, hi[0].x, hi[0].y);
#pragma unroll
            for (int c = 1; c < CS; ++c)
                if (c < cs) { s.x += lo[c].x; s.y += lo[c].y; s.z += hi[c].x; s.w += hi[c].y; }
        } else {
            s = tile_sum[il];
        }
        const int i = tile0 + il;
        if (i >= a.n_i) continue;
        if (n_groups == 1) {                                           // a6: epilogue
            a.acc[3 * (size_t)i + 0] = (float)s.x;
            a.acc[3 * (size_t)i + 1] = (float)s.y;
            a.acc[3 * (size_t)i + 2] = (float)s.z;
            if (a.pot) a.pot[i] = -(float)s.w;
        } else {
            a.partial[(size_t)i * n_groups + group] = s;          // [n_i][n_groups]: a particle's partials are contiguous
        }
    }
    if (CS > 1) cluster_sync_all();                                    // nobody leaves while its shared memory is being read
    NB_STAMP(3);

    // a7, level 4 (S > CS): FP64 cluster partials in global memory; the CTA that arrives LAST at the ticket of its
    // (i-tile, slice) sums them in the order group = 0 .. S/CS-1 and leaves the ticket at zero for the next call.
    if (n_groups > 1) {
        // Release / acquire through ONE thread: the barrier orders every thread's partial stores before thread 0's
        // atom.acq_rel at GPU scope (cumulative), and the last CTA's loads after the second barrier come after it -- no
        // __threadfence by all threads (a MEMBAR per thread: ~1 us each side, measured with %globaltimer stamps).
        __shared__ int s_last;
        __syncthreads();
        if (threadIdx.x == 0) {
            int* tk = a.tickets + blockIdx.x * cs + rank;
            int ticket;
            asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(ticket) : "l"(tk) : "memory");
            s_last = (ticket == n_groups - 1);
            if (s_last) *tk = 0;
        }
        __syncthreads();
        NB_STAMP(4);
        if (!s_last) return;
        // One thread per (i, half): half = (ax, ay) or (az, phi); the loads run ahead, the adds keep the order g = 0 .. n-1.
        // (One SM pulls the other CTAs' partials at only ~25-40 GB/s, whatever the number of loads in flight -- 1.5 us for
        // 18 groups of a 64-particle tile, 3.9 us for 37 groups of 128, against 0.8-1.0 us when every load hits the SM's own
        // row; waiting 3 us first changes nothing (measured with %globaltimer stamps).  The planner keeps groups x tile small.)
        for (int t = threadIdx.x; t < 2 * SLICE; t += kSmallThreads) {
            const int i = tile0 + (int)rank * SLICE + (t >> 1), half = t & 1;
            if (i >= a.n_i) continue;
            const double2* p2 = reinterpret_cast<const double2*>(a.partial + (size_t)i * n_groups) + half;
            double2 sum = __ldcg(p2);
#pragma unroll 8
            for (int g = 1; g < n_groups; ++g) {
                const double2 v = __ldcg(p2 + 2 * g);
                sum.x += v.x; sum.y += v.y;
            }
            if (half == 0) {
                a.acc[3 * (size_t)i + 0] = (float)sum.x;
                a.acc[3 * (size_t)i + 1] = (float)sum.y;
            } else {
                a.acc[3 * (size_t)i + 2] = (float)sum.x;
                if (a.pot) a.pot[i] = -(float)sum.y;
            }
        }
        NB_STAMP(5);
    }
}

}  // namespace nb
