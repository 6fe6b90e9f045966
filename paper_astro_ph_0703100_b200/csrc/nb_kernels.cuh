// nb_kernels.cuh -- sm_100a device code for the all-pairs softened gravity path.
//
// Rows of SURVEY.md section 8(a) implemented here (citations: PAPER.md by line):
//   a1  j-pack            nb_pack_j_kernel         Fig. A.1 packing loop
//   a2  j-tile staging    TMA bulk copy + mbarrier ring in nb_force_kernel   step (d) J-PACKING
//   a3  i-load            prologue of nb_force_kernel                        step (e)
//   a4  pair interaction  pair_body()                                        step (h); Eq. (1); Fig. A.3 PAPER.md:458-471;
//                                                                            potential Fig. A.4
//   a5  two-level sum     per-tile partial -> running total                  steps (f),(g),(i); Eq. (2)
//   a6  epilogue          end of nb_force_kernel / nb_reduce_kernel          step (i)
//   a7  j-split + reduce  WJ (warps) and S (CTAs) split, fixed-order sums    (paper analogue: force-memory round trips)
//
// Layout of the packed j-array: one 16-byte record (x, y, z, m) per j-particle -- the paper's own
// [n_j][JDIM = 4] rows -- in a 128-byte aligned array, so that a tile is one
// contiguous 1-D TMA bulk copy and one broadcast LDS.128 yields a whole j-particle.
//
// Register layout of the i-particles: each thread owns K i-particles as K/2 PAIRS held in 64-bit
// registers, so that the packed FP32 instructions (add/mul/fma.f32x2 -> SASS FADD2/FMUL2/FFMA2)
// process two i-particles against one j-particle per instruction; the j operand is the 32-bit
// broadcast form of those instructions.  Why: on sm_100 the loop is bound
// by register-file read bandwidth and issue slots, not by the FMA pipe alone; the packed forms halve
// the issue slots and the scalar j operand saves a register read per instruction.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nb_packed.cuh"

namespace nb {

// ---------------------------------------------------------------- a1: j-pack
// One thread per j-particle: (x, y, z) || m -> float4.
__global__ void __launch_bounds__(256) nb_pack_j_kernel(const float* __restrict__ x_j, const float* __restrict__ m_j,
                                                        int n_j, float4* __restrict__ jp) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_j) return;
    jp[j] = make_float4(x_j[3 * (size_t)j + 0], x_j[3 * (size_t)j + 1], x_j[3 * (size_t)j + 2], m_j[j]);
}

// ---------------------------------------------------------------- a4: two i-particles x one j-particle
// 13 packed FP32-pipe instructions (3 FADD2, 3 FFMA2, 3 FMUL2, 3 FFMA2, 1 FADD2) + 2 MUFU.RSQ.
// nxi = (-x_i0, -x_i1) etc., so d = r_j - r_i.  xj, yj, zj, mj hold the j value in both halves.
//
// Coincident pairs (reading R1: all three differences exactly zero => the pair adds nothing).
//   MASK_EXACT : test (dx | dy | dz) == 0 bitwise and send r2 to +inf, so rsqrt gives +0 and every
//                term of the pair vanishes; 2 ALU-pipe instructions with 4 register reads per pair.
//   MASK_NONE  : no masking; valid for a block of j-particles that is known (from the coincidence lists built
//                by nb_coin_probe_kernel) to hold no partner of this warp's i-particles, where it gives bit for
//                bit what MASK_EXACT gives -- and everywhere when phi is not wanted and eps2 >= 2^-40, because an
//                unmasked coincident pair adds m u^3 * (+-0) = +-0 to a.  13 + 1 instructions.
// (A third, speculative variant -- flag r2 == eps2 in the loop, redo a flagged 256-j block with the mask -- was the
//  default earlier in this round and was removed: DESIGN.md section 10.)
// PHI = false: the caller does not want the potential (pot_out == NULL): 12 FP32-pipe instructions per pair.
template <int MASK, bool PHI = true>
__device__ __forceinline__ void pair_body(u64 xj, u64 yj, u64 zj, u64 mj, u64 nxi, u64 nyi, u64 nzi, u64 eps2_2,
                                          u64& ax, u64& ay, u64& az, u64& ph) {
    const u64 dx = add2(xj, nxi);                    // dx = xj - xi
    const u64 dy = add2(yj, nyi);
    const u64 dz = add2(zj, nzi);
    u64 r2 = fma2(dx, dx, eps2_2);                   // r2 = dx2+dy2+dz2+eps2 PAPER.md:464
    r2 = fma2(dy, dy, r2);
    r2 = fma2(dz, dz, r2);
    float r2a, r2b;
    unpack2(r2, r2a, r2b);
    if (MASK == MASK_EXACT) {
        // coincident <=> all three differences are exactly +0 (x - x rounds to +0)
        const float inf = __int_as_float(0x7f800000);
        float dxa, dxb, dya, dyb, dza, dzb;
        unpack2(dx, dxa, dxb); unpack2(dy, dya, dyb); unpack2(dz, dza, dzb);
        const uint32_t ta = __float_as_uint(dxa) | __float_as_uint(dya) | __float_as_uint(dza);
        const uint32_t tb = __float_as_uint(dxb) | __float_as_uint(dyb) | __float_as_uint(dzb);
        r2a = (ta == 0u) ? inf : r2a;                // rsqrt(+inf) = +0 -> the pair adds exactly 0
        r2b = (tb == 0u) ? inf : r2b;
    }
    const u64 u = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));   // r1i = 1/sqrt(r2)
    const u64 u2 = mul2(u, u);                       // r2i
    const u64 mu = mul2(mj, u);                      // pot = mj * r1i
    const u64 mu3 = mul2(mu, u2);                    // mr3i
    ax = fma2(mu3, dx, ax);                          // OUTPUT[0..2] += mr3i*d PAPER.md:469-471
    ay = fma2(mu3, dy, ay);
    az = fma2(mu3, dz, az);
    if (PHI) ph = add2(ph, mu);                      // OUTPUT[6] -= pot (sign applied at the end) PAPER.md:552
}

// One tile: K/2 i-pairs of this thread against np j-particles in shared memory; partial sums start from zero (Eq. (2)).
// EPS_I (row f3): the softening is a property of the i-particle (Fig. A.1) and sits, packed, in e2[].
// ACC = true: the partial sums continue (the caller zeroed them; row f2 sweeps one Eq. (2) block in several parts).
template <int K, int MASK, bool EPS_I = false, bool PHI = true, bool ACC = false>
__device__ __forceinline__ void tile_sweep(const float4* __restrict__ sp, int np, const u64 (&nxi)[K / 2], const u64 (&nyi)[K / 2],
                                           const u64 (&nzi)[K / 2], u64 eps2_2, u64 (&pax)[K / 2], u64 (&pay)[K / 2],
                                           u64 (&paz)[K / 2], u64 (&pph)[K / 2], const u64 (&e2)[K / 2]) {
    if (!ACC) {
#pragma unroll
        for (int k = 0; k < K / 2; ++k) { pax[k] = 0ull; pay[k] = 0ull; paz[k] = 0ull; pph[k] = 0ull; }
    }
#pragma unroll 4
    for (int j = 0; j < np; ++j) {
        const float4 J = sp[j];                                        // broadcast LDS.128: x y z m
        const u64 xj = pack2(J.x, J.x), yj = pack2(J.y, J.y), zj = pack2(J.z, J.z), mj = pack2(J.w, J.w);
#pragma unroll
        for (int k = 0; k < K / 2; ++k)
            pair_body<MASK, PHI>(xj, yj, zj, mj, nxi[k], nyi[k], nzi[k], EPS_I ? e2[k] : eps2_2, pax[k], pay[k], paz[k], pph[k]);
    }
}

// ---------------------------------------------------------------- coincidence lists (reading R1, large calls)
// For large calls the coincident pairs (reading R1) are located BEFORE the force kernel by
// a hash join on the positions, so that the hot loop carries no test at all (MASK_NONE) and only the
// few (i-group, j-segment) combinations that do hold a coincident pair run the masked loop:
//   nb_coin_insert_kernel : every j-particle is entered in an open-addressing table keyed by its
//                           canonical position bits (subnormals and -0 -> +0, as add.ftz sees them);
//   nb_coin_probe_kernel  : one CTA per i-group (the 32*K i-particles one warp of the force kernel
//                           owns) looks its i-particles up and writes the sorted list of j-SEGMENTS
//                           (kCoinSeg consecutive j, global index / kCoinSeg) that hold a partner.
// List layout: int [n_groups][1 + kCoinCap] = (count, segment ids ascending); count = -1 means "too
// many, mask every block".  *flag != 0 means the table degenerated (very many identical positions):
// the force kernel then masks everywhere.  Either way the stored result equals the always-masked one.
constexpr int kCoinSeg = 256;         // j-particles per segment (= SUB of the force kernel)
constexpr int kCoinSegShift = 8;
constexpr int kCoinCap = 8;           // segments kept per i-group
constexpr int kCoinRaw = 32;          // distinct segments collected per i-group before giving up (set of 64 slots)
constexpr int kCoinMaxProbe = 2048;   // probe steps before giving up

// table entries: 0 = empty, else j + 1
// stride = float4 per j record (1 for the force path, 2 for the force + jerk path)
__global__ void __launch_bounds__(256) nb_coin_insert_kernel(const float4* __restrict__ jp, int stride, int n_j,
                                                             uint32_t* __restrict__ table, uint32_t mask,
                                                             int* __restrict__ flag) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_j) return;
    const float4 J = jp[(size_t)j * stride];
    uint32_t slot = coin_hash(coin_canon(J.x), coin_canon(J.y), coin_canon(J.z)) & mask;
    for (int step = 0; step < kCoinMaxProbe; ++step) {
        if (table[slot] == 0u && atomicCAS(table + slot, 0u, (uint32_t)j + 1u) == 0u) return;
        slot = (slot + 1u) & mask;
    }
    *flag = 1;                                                         // degenerate input: mask everywhere
}

__global__ void __launch_bounds__(256) nb_coin_probe_kernel(const float* __restrict__ x_i, int n_i,
                                                            const float4* __restrict__ jp, int stride,
                                                            const uint32_t* __restrict__ table, uint32_t mask,
                                                            int* __restrict__ lists) {
    __shared__ int set[2 * kCoinRaw];                                  // open-addressing set of segment ids, -1 = empty
    __shared__ int n_set;
    __shared__ int overflow;
    if (threadIdx.x < 2 * kCoinRaw) set[threadIdx.x] = -1;
    if (threadIdx.x == 0) { n_set = 0; overflow = 0; }
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;               // blockDim.x = 32 * K = one i-group
    if (i < n_i) {
        const uint32_t cx = coin_canon(x_i[3 * (size_t)i + 0]), cy = coin_canon(x_i[3 * (size_t)i + 1]), cz = coin_canon(x_i[3 * (size_t)i + 2]);
        uint32_t slot = coin_hash(cx, cy, cz) & mask;
        int step = 0;
        for (; step < kCoinMaxProbe; ++step) {
            const uint32_t e = table[slot];
            if (e == 0u) break;
            const float4 J = jp[(size_t)(e - 1u) * stride];
            if (coin_canon(J.x) == cx && coin_canon(J.y) == cy && coin_canon(J.z) == cz) {
                const int seg = (int)((e - 1u) >> kCoinSegShift);
                uint32_t h = ((uint32_t)seg * 2654435761u) >> 26;      // 64 slots
                bool placed = false;
                for (int q = 0; q < 2 * kCoinRaw && !placed; ++q) {
                    const int old = atomicCAS(&set[h], -1, seg);
                    if (old == seg) placed = true;
                    else if (old == -1) { placed = true; if (atomicAdd(&n_set, 1) >= kCoinRaw) overflow = 1; }
                    h = (h + 1u) & (2 * kCoinRaw - 1);
                }
                if (!placed) overflow = 1;
                if (*(volatile int*)&overflow) break;
            }
            slot = (slot + 1u) & mask;
        }
        if (step == kCoinMaxProbe) overflow = 1;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int* out = lists + (size_t)blockIdx.x * (1 + kCoinCap);
        int n = 0, cnt = 0;
        int seg[2 * kCoinRaw];
        for (int q = 0; q < 2 * kCoinRaw; ++q)
            if (set[q] >= 0) seg[n++] = set[q];
        for (int a = 1; a < n; ++a) {                                  // insertion sort of <= 64 distinct entries
            const int v = seg[a];
            int b = a - 1;
            while (b >= 0 && seg[b] > v) { seg[b + 1] = seg[b]; --b; }
            seg[b + 1] = v;
        }
        const bool too_many = (overflow != 0) || n > kCoinCap;
        for (int q = 0; q < n && !too_many; ++q) out[1 + cnt++] = seg[q];
        out[0] = too_many ? -1 : cnt;
    }
}

struct ForceArgs {
    const float* x_i;      // [n_i][3]
    const float* eps2_i;   // EPS_I: [n_i] softening squared of every i-particle
    const float4* jp;      // packed j records (x, y, z, m)
    const float* xj_raw;   // non-null (with mj_raw): small call, every warp group packs its own j sub-range straight
    const float* mj_raw;   //   from x_j / m_j into its ring (it fits whole) -- no nb_pack_j_kernel launch, no TMA
    float* acc;            // [n_i][3]
    float* pot;            // [n_i] or nullptr
    double4* partial;      // [S][n_i] when S > 1
    int* tickets;          // [tiles_i] zero between calls; non-null => the last CTA of an i-tile sums the partials
    const int* coin_lists; // MODE_LIST: [n_groups][1 + kCoinCap]
    const int* coin_flag;  // MODE_LIST: != 0 -> mask everywhere
    const int* i_off;      // nb_batched_kernel: [n_batch + 1] first i of every sub-problem
    const int* j_off;      // nb_batched_kernel: [n_batch + 1] first j of every sub-problem
    const int* tile_start; // nb_batched_kernel: [n_batch + 1] first CTA of every sub-problem (exclusive scan of its i-tiles)
    const int* cta_batch;  // nb_batched_kernel: [number of CTAs] sub-problem of every CTA
    const int* j_index;    // nb_batched_kernel<INDEXED>: [n_list_total] indices into jp (the packed particle array)
    int n_batch;
    int n_i;
    int n_j;
    int S;
    float eps2;
};

// how the force kernel honours the coincident-pair rule
enum { MODE_EXACT = 0,     // masked loop everywhere (eps2 == 0 or tiny; per-i softening on small calls)
       MODE_BLOOM = 1,     // per-warp Bloom filter of the i-positions in shared memory, every 256-j block tested (mid-size calls)
       MODE_LIST = 2 };    // coincidence lists from the pre-pass, no test in the hot loop (large calls; a-only calls)

// ---------------------------------------------------------------- a2..a7: the force kernel
// CTA = 8 warps = WI (along i) x WJ (along j).  A CTA owns 32*K*WI i-particles (K per thread, in
// registers) and the S-th part (blockIdx.y) of the j-range, which is cut again into WJ sub-ranges.
// Each sub-range is streamed through its own shared-memory ring by 1-D TMA bulk copies issued by
// lane 0 of the group's first warp; "full" mbarriers count bytes, "empty" mbarriers count the WI
// consuming warps.
template <int K, int WI, int WJ, int TJ, int STAGES, int MODE, bool EPS_I = false, bool PHI = true, bool DIRECT = false,
          int SUB = 256>
__global__ void __launch_bounds__(32 * WI * WJ, 1) nb_force_kernel(const ForceArgs a) {
    static_assert(K % 2 == 0, "i-particles are held in pairs");
    static_assert(MODE == MODE_EXACT || MODE == MODE_BLOOM || MODE == MODE_LIST, "masked everywhere, Bloom filter, or coincidence lists");
    static_assert(SUB == kCoinSeg, "coincidence segments are SUB j-particles");
    extern __shared__ __align__(128) unsigned char smem_raw[];

    // i-range [i_lo, i_hi) this CTA draws its tile from, j-range [jr_lo, jr_lo + jr_n) it sums over
    const int i_lo = blockIdx.x * (32 * K * WI), i_hi = a.n_i, jr_lo = 0, jr_n = a.n_j;
    constexpr int RING_BYTES = STAGES * TJ * 16;
    unsigned char* rings = smem_raw;                                   // [WJ][STAGES][TJ] float4
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

    // j sub-range of this warp group
    const long long G = (long long)a.S * WJ;
    const long long g = (long long)blockIdx.y * WJ + wj;
    const int j_begin = jr_lo + (int)((long long)jr_n * g / G);
    const int j_end = jr_lo + (int)((long long)jr_n * (g + 1) / G);
    const int n_sub = j_end - j_begin;
    const int n_tiles = (n_sub + TJ - 1) / TJ;
    const unsigned char* src = reinterpret_cast<const unsigned char*>(a.jp + j_begin);

    // a3: i-particles of this thread (clamped loads; stores are guarded), pair k2 = (k = 2 k2, 2 k2 + 1)
    // a warp owns 32*K consecutive i-particles, so that an aliased i-set meets its own copies in few j-tiles
    const int i_base = i_lo + wi * (32 * K) + lane;
    u64 nxi[K / 2], nyi[K / 2], nzi[K / 2];
#pragma unroll
    for (int k2 = 0; k2 < K / 2; ++k2) {
        const int i0 = min(i_base + (2 * k2) * 32, i_hi - 1);
        const int i1 = min(i_base + (2 * k2 + 1) * 32, i_hi - 1);
        nxi[k2] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 0]), neg_canon(a.x_i[3 * (size_t)i1 + 0]));
        nyi[k2] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 1]), neg_canon(a.x_i[3 * (size_t)i1 + 1]));
        nzi[k2] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 2]), neg_canon(a.x_i[3 * (size_t)i1 + 2]));
    }
    const u64 eps2_2 = pack2(a.eps2, a.eps2);
    u64 e2[K / 2];
#pragma unroll
    for (int k2 = 0; k2 < K / 2; ++k2) {
        if (EPS_I) {
            const int i0 = min(i_base + (2 * k2) * 32, i_hi - 1);
            const int i1 = min(i_base + (2 * k2 + 1) * 32, i_hi - 1);
            e2[k2] = pack2(a.eps2_i[i0], a.eps2_i[i1]);
        } else {
            e2[k2] = eps2_2;
        }
    }

    // MODE_BLOOM: the filter of this warp's i-positions (the WJ warps with the same wi share it)
    uint32_t* filt = reinterpret_cast<uint32_t*>(smem_raw + WJ * RING_BYTES + 2 * WJ * STAGES * 8) + wi * kBloomWords;
    if (MODE == MODE_BLOOM) {
        uint4* z = reinterpret_cast<uint4*>(smem_raw + WJ * RING_BYTES + 2 * WJ * STAGES * 8);
        for (int q = threadIdx.x; q < WI * kBloomWords / 4; q += 32 * WI * WJ) z[q] = make_uint4(0u, 0u, 0u, 0u);
        __syncthreads();
        if (wj == 0) {
#pragma unroll
            for (int k = 0; k < K; ++k) {
                const int i = min(i_base + k * 32, i_hi - 1);
                bloom_set(filt, bloom_key(a.x_i[3 * (size_t)i + 0], a.x_i[3 * (size_t)i + 1], a.x_i[3 * (size_t)i + 2]));
            }
        }
    }
    __syncthreads();                                                   // barriers initialised, filters built

    // Small calls (nbody_b200.cu: the whole sub-range fits the ring): rows a1 + a2 in one step -- the WI warps of the
    // group pack their sub-range from x_j / m_j into the ring themselves (Fig. A.1 packing loop);
    // tile t then sits in slot t, exactly where the TMA path would have put it.
    constexpr bool direct = DIRECT;                                    // a template parameter: the large-call kernels carry none of this
    if (direct) {
        float4* rp = reinterpret_cast<float4*>(rings + wj * RING_BYTES);
        for (int q = wi * 32 + lane; q < n_sub; q += WI * 32) {
            const size_t j = (size_t)(j_begin + q);
            rp[q] = make_float4(a.xj_raw[3 * j + 0], a.xj_raw[3 * j + 1], a.xj_raw[3 * j + 2], a.mj_raw[j]);
        }
        __syncthreads();
    } else if (producer) {
        const int pre = n_tiles < STAGES ? n_tiles : STAGES;
        for (int t = 0; t < pre; ++t) {
            const uint32_t bytes = (uint32_t)min(TJ, n_sub - t * TJ) * 16u;
            mbar_expect_tx(full0 + 8 * t, bytes);
            tma_load_1d(ring + t * TJ * 16, src + (size_t)t * TJ * 16, bytes, full0 + 8 * t);
        }
    }

    double run[K][4];                                                  // running totals (outer level of Eq. (2))
#pragma unroll
    for (int k = 0; k < K; ++k) { run[k][0] = run[k][1] = run[k][2] = run[k][3] = 0.0; }

    // MODE_LIST: ascending j-segments that hold a partner of this warp's i-particles (warp-uniform)
    const int* coin = nullptr;
    int coin_cnt = 0, coin_pos = 0, coin_next = 0x7fffffff;
    if (MODE == MODE_LIST && a.coin_lists != nullptr) {               // nullptr: no block needs the mask (see nbody_b200.cu)
        coin = a.coin_lists + (size_t)(blockIdx.x * WI + wi) * (1 + kCoinCap);
        coin_cnt = (*a.coin_flag != 0) ? -1 : coin[0];
        if (coin_cnt > 0) coin_next = coin[1];
    }

    for (int t = 0; t < n_tiles; ++t) {
        const int slot = t % STAGES;
        const uint32_t parity = (uint32_t)(t / STAGES) & 1u;
        if (!direct) mbar_wait(full0 + 8 * slot, parity);

        const int np = min(TJ, n_sub - t * TJ);
        const float4* sp = reinterpret_cast<const float4*>(rings + wj * RING_BYTES + slot * TJ * 16);

        // Eq. (2) blocks of at most SUB consecutive j: partial sums from zero, then added to the running total
        for (int c = 0; c < np; c += SUB) {
            const int nc = min(SUB, np - c);
            u64 pax[K / 2], pay[K / 2], paz[K / 2], pph[K / 2];
            if (MODE == MODE_LIST) {
                const int j0 = j_begin + t * TJ + c;                   // global index of the block's first j
                const int seg_lo = j0 >> kCoinSegShift, seg_hi = (j0 + nc - 1) >> kCoinSegShift;
                while (coin_next < seg_lo) {
                    ++coin_pos;
                    coin_next = (coin_pos < coin_cnt) ? coin[1 + coin_pos] : 0x7fffffff;
                }
                if (coin_cnt < 0 || coin_next <= seg_hi)               // rare: the block holds a coincident pair
                    tile_sweep<K, MASK_EXACT, EPS_I, PHI>(sp + c, nc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph, e2);
                else
                    tile_sweep<K, MASK_NONE, EPS_I, PHI>(sp + c, nc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph, e2);
            } else if (MODE == MODE_BLOOM) {
                bool hit = false;                                      // may a j of this block coincide with an i of this warp?
#pragma unroll
                for (int q = 0; q < SUB; q += 32) {                    // branch-free: 8 independent chains (a short block tests its last j again)
                    const float4 J = sp[c + min(q + lane, nc - 1)];
                    hit |= bloom_test(filt, bloom_key(J.x, J.y, J.z));
                }
                if (__any_sync(0xffffffffu, hit))
                    tile_sweep<K, MASK_EXACT, EPS_I, PHI>(sp + c, nc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph, e2);
                else
                    tile_sweep<K, MASK_NONE, EPS_I, PHI>(sp + c, nc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph, e2);
            } else {
                tile_sweep<K, MASK_EXACT, EPS_I, PHI>(sp + c, nc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph, e2);
            }
            // a5: block partial -> running total
#pragma unroll
            for (int k2 = 0; k2 < K / 2; ++k2) {
                float lo, hi;
                unpack2(pax[k2], lo, hi); run[2 * k2][0] += (double)lo; run[2 * k2 + 1][0] += (double)hi;
                unpack2(pay[k2], lo, hi); run[2 * k2][1] += (double)lo; run[2 * k2 + 1][1] += (double)hi;
                unpack2(paz[k2], lo, hi); run[2 * k2][2] += (double)lo; run[2 * k2 + 1][2] += (double)hi;
                if (PHI) { unpack2(pph[k2], lo, hi); run[2 * k2][3] += (double)lo; run[2 * k2 + 1][3] += (double)hi; }
            }
        }

        // release the slot; the producer refills it with tile t' + STAGES.  With several consumer
        // warps the refill trails by one tile so that the producer rarely waits for a slower warp.
        __syncwarp();
        if (direct) continue;
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
        if (producer) {
            const int tt = (WI > 1) ? t - 1 : t;
            if (tt >= 0 && tt + STAGES < n_tiles) {
                const int rs = tt % STAGES;
                mbar_wait(empty0 + 8 * rs, (uint32_t)(tt / STAGES) & 1u);
                const int tn = tt + STAGES;
                const uint32_t bytes = (uint32_t)min(TJ, n_sub - tn * TJ) * 16u;
                mbar_expect_tx(full0 + 8 * rs, bytes);
                tma_load_1d(ring + rs * TJ * 16, src + (size_t)tn * TJ * 16, bytes, full0 + 8 * rs);
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
        if (wj == 0) {
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
    }

    // a6: epilogue
    if (wj == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const int i = i_base + k * 32;
            if (i >= i_hi) continue;
            if (a.S == 1) {
                a.acc[3 * (size_t)i + 0] = (float)run[k][0];
                a.acc[3 * (size_t)i + 1] = (float)run[k][1];
                a.acc[3 * (size_t)i + 2] = (float)run[k][2];
                if (a.pot) a.pot[i] = -(float)run[k][3];
            } else {
                a.partial[(size_t)blockIdx.y * a.n_i + i] = make_double4(run[k][0], run[k][1], run[k][2], run[k][3]);
            }
        }
    }

    // a7 (inter-CTA), fused: the CTA that finishes LAST among the S chunks of this i-tile sums the S partials in the
    // fixed order s = 0 .. S-1 (so the result does not depend on which CTA that is) and writes a and phi.  The
    // ticket counter of the tile returns to zero for the next call.  (nb_reduce_kernel is the same sum as a separate
    // launch; it is kept for the NB_FUSED_REDUCE=0 comparison.)
    if (a.S > 1 && a.tickets != nullptr) {
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
            const double2* p2 = reinterpret_cast<const double2*>(a.partial + i);          // L2 reads (other SMs wrote these)
            double2 lo = __ldcg(p2), hi = __ldcg(p2 + 1);
            double4 sum = make_double4(lo.x, lo.y, hi.x, hi.y);
#pragma unroll 8
            for (int c = 1; c < a.S; ++c) {                            // loads run ahead, the adds keep the order s = 0 .. S-1
                p2 = reinterpret_cast<const double2*>(a.partial + (size_t)c * a.n_i + i);
                lo = __ldcg(p2); hi = __ldcg(p2 + 1);
                sum.x += lo.x; sum.y += lo.y; sum.z += hi.x; sum.w += hi.y;
            }
            a.acc[3 * (size_t)i + 0] = (float)sum.x;
            a.acc[3 * (size_t)i + 1] = (float)sum.y;
            a.acc[3 * (size_t)i + 2] = (float)sum.z;
            if (a.pot) a.pot[i] = -(float)sum.w;
        }
    }
}

// f2: exclusive scan of the i-tiles per sub-problem -> first CTA of every sub-problem (one CTA, n_batch + 1 outputs)
__global__ void __launch_bounds__(1024) nb_batch_scan_kernel(const int* __restrict__ i_off, int n_batch, int tile_i,
                                                             int* __restrict__ tile_start, int* __restrict__ cta_batch) {
    __shared__ int warp_sum[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int base = 0; base < n_batch; base += 1024) {
        const int b = base + threadIdx.x;
        const int tiles = (b < n_batch) ? (max(i_off[b + 1] - i_off[b], 0) + tile_i - 1) / tile_i : 0;
        int incl = tiles;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += v;
        }
        if (lane == 31) warp_sum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int w = warp_sum[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, w, d);
                if (lane >= d) w += v;
            }
            warp_sum[lane] = w;                                        // inclusive over warps
        }
        __syncthreads();
        const int before = carry + (warp > 0 ? warp_sum[warp - 1] : 0) + incl - tiles;
        if (b < n_batch) {
            tile_start[b] = before;
            for (int t = 0; t < tiles; ++t) cta_batch[before + t] = b;
        }
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + tiles;
        __syncthreads();
    }
    if (threadIdx.x == 0) tile_start[n_batch] = carry;
}

// a7 (inter-CTA): second pass, fixed-order sum over the S chunk partials
__global__ void __launch_bounds__(128) nb_reduce_kernel(const double4* __restrict__ partial, int n_i, int S,
                                                        float* __restrict__ acc, float* __restrict__ pot) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_i) return;
    double4 s = partial[i];
#pragma unroll 8
    for (int c = 1; c < S; ++c) {                                      // loads run ahead, the adds keep the order
        const double4 v = partial[(size_t)c * n_i + i];
        s.x += v.x; s.y += v.y; s.z += v.z; s.w += v.w;
    }
    acc[3 * (size_t)i + 0] = (float)s.x;
    acc[3 * (size_t)i + 1] = (float)s.y;
    acc[3 * (size_t)i + 2] = (float)s.z;
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
