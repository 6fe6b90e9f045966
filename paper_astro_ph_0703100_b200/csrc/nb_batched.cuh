// nb_batched.cuh -- sm_100a kernel of row f2: many small (i-set, j-set) sub-problems of Eq. (1) in ONE launch,
// the call pattern of a host tree code with interaction lists of "several thousands" particles
// (PAPER.md:246 last sentence; section 4.4).
//
// One CTA = 8 warps works on up to 64 G i-particles of ONE sub-problem (G = 1, 2 or 4 packed groups of 64, a
// template parameter).  Unlike nb_force_kernel every warp holds the SAME i-particles (in registers) and the 8 warps
// split the j-list, each streaming its part through its own TMA + mbarrier ring; nothing leaves the CTA but a_i, phi_i.
//   - K per CTA at run time: a tile that holds n_i <= 64 / 128 / 192 / 256 particles runs 1 / 2 / 3 / 4 packed groups
//     (tile_sweep<2 KG>), so the padding of a sub-problem is at most 63 idle lanes;
//   - coincident pairs (reading R1): interaction lists contain the group's own members, so EVERY
//     sub-problem has them -- but only where a j-particle lies inside the bounding box of the tile's i-particles.
//     MASKED = true tests the list kBatchSub j at a time against that box: a part with a j inside runs the masked
//     loop, the others the untested loop (bit for bit the same there).  MASKED = false (phi not wanted and
//     eps2 >= 2^-40: an unmasked coincident pair adds +-0 to a) runs the untested loop everywhere, no test.
// Measured on the T1 tree lists: G = 1 is the fastest shape (66 % of roofline: 83 % lane use x 80 % loop
// efficiency; 60 % with every pair masked).  A flag-only loop with the flagged blocks redone by all 8 warps together
// was tried and removed (55 %: the redo serialises the CTA).
#pragma once
#include "nb_kernels.cuh"

namespace nb {

constexpr int kBatchSub = 64;        // j-particles per bounding-box test (a multiple of 32, divides the 256-j tile)

template <int KG, int G>
__device__ __forceinline__ const u64 (&first_groups(const u64 (&arr)[G]))[KG] {
    return *reinterpret_cast<const u64(*)[KG]>(&arr[0]);
}
template <int KG, int G>
__device__ __forceinline__ u64 (&first_groups(u64 (&arr)[G]))[KG] {
    return *reinterpret_cast<u64(*)[KG]>(&arr[0]);
}

// the first KG packed groups against np j-particles; the partial sums CONTINUE (the caller zeroes them per Eq. (2) block)
template <int KG, int MASK, bool PHI, int G>
__device__ __forceinline__ void sweep_groups(const float4* __restrict__ sp, int np, const u64 (&nxi)[G], const u64 (&nyi)[G],
                                             const u64 (&nzi)[G], u64 eps2_2, u64 (&pax)[G], u64 (&pay)[G],
                                             u64 (&paz)[G], u64 (&pph)[G]) {
    tile_sweep<2 * KG, MASK, false, PHI, true>(sp, np, first_groups<KG, G>(nxi), first_groups<KG, G>(nyi),
                                               first_groups<KG, G>(nzi), eps2_2, first_groups<KG, G>(pax),
                                               first_groups<KG, G>(pay), first_groups<KG, G>(paz),
                                               first_groups<KG, G>(pph), first_groups<KG, G>(nxi) /* e2: unused */);
}

// kg (1..G) active packed groups, uniform over the CTA; the inactive groups' partial sums stay zero
template <int MASK, bool PHI, int G>
__device__ __forceinline__ void sweep_dyn(int kg, const float4* __restrict__ sp, int np, const u64 (&nxi)[G], const u64 (&nyi)[G],
                                          const u64 (&nzi)[G], u64 eps2_2, u64 (&pax)[G], u64 (&pay)[G],
                                          u64 (&paz)[G], u64 (&pph)[G]) {
    if (G >= 4 && kg >= 4) sweep_groups<(G >= 4 ? 4 : 1), MASK, PHI, G>(sp, np, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
    else if (G >= 3 && kg == 3) sweep_groups<(G >= 3 ? 3 : 1), MASK, PHI, G>(sp, np, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
    else if (G >= 2 && kg == 2) sweep_groups<(G >= 2 ? 2 : 1), MASK, PHI, G>(sp, np, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
    else sweep_groups<1, MASK, PHI, G>(sp, np, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
}

template <int G>
__device__ __forceinline__ void add_partials(double (&run)[2 * G][4], const u64 (&pax)[G], const u64 (&pay)[G], const u64 (&paz)[G],
                                             const u64 (&pph)[G]) {
#pragma unroll
    for (int k2 = 0; k2 < G; ++k2) {
        float lo, hi;
        unpack2(pax[k2], lo, hi); run[2 * k2][0] += (double)lo; run[2 * k2 + 1][0] += (double)hi;
        unpack2(pay[k2], lo, hi); run[2 * k2][1] += (double)lo; run[2 * k2 + 1][1] += (double)hi;
        unpack2(paz[k2], lo, hi); run[2 * k2][2] += (double)lo; run[2 * k2 + 1][2] += (double)hi;
        unpack2(pph[k2], lo, hi); run[2 * k2][3] += (double)lo; run[2 * k2 + 1][3] += (double)hi;
    }
}

// A tile that holds at most 32 particles (the ragged tail of a group) would leave one half of every packed
// instruction idle.  It packs over j instead: both halves carry the SAME i-particle, the two halves of the j operand
// are two consecutive j-particles, and the two half-sums are added at the end -- the tile takes half the time.
// The sums CONTINUE (the caller zeroes them per Eq. (2) block); np is even except for the last part of a list.
template <int MASK, bool PHI>
__device__ __forceinline__ void half_sweep(const float4* __restrict__ sp, int np, u64 nx, u64 ny, u64 nz, u64 eps2_2, u64& ax,
                                           u64& ay, u64& az, u64& ph) {
    int j = 0;
#pragma unroll 4
    for (; j + 2 <= np; j += 2) {
        const float4 A = sp[j], B = sp[j + 1];
        pair_body<MASK, PHI>(pack2(A.x, B.x), pack2(A.y, B.y), pack2(A.z, B.z), pack2(A.w, B.w), nx, ny, nz, eps2_2, ax, ay, az, ph);
    }
    if (j < np) {                                                      // odd tail: the partner is a massless particle far away
        const float4 A = sp[j];
        const float far = 3.0e18f;
        pair_body<MASK, PHI>(pack2(A.x, far), pack2(A.y, far), pack2(A.z, far), pack2(A.w, 0.0f), nx, ny, nz, eps2_2, ax, ay, az, ph);
    }
}

// 16-byte asynchronous copy global -> shared (LDGSTS) and its group bookkeeping: the gathered ring fill of INDEXED lists
__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// G = packed groups of 64 i-particles a CTA can hold (tile = 64 G); STAGES = ring depth per warp.
// INDEXED: the lists are int32 indices (a.j_index) into ONE array of packed particle records (a.jp) -- what a tree code
// holds: 4 bytes per list entry instead of 16.  A ring slot is then filled by 256 gathered 16-byte cp.async copies (8 per
// lane, the indices of the tile after next already in registers) instead of one bulk copy; completion is tracked per lane
// with cp.async groups (one group per tile, empty ones included, so the count is uniform) + __syncwarp.
template <bool MASKED, int G, int STAGES, bool INDEXED = false>
__global__ void __launch_bounds__(256, (G == 1 ? 2 : 1)) nb_batched_kernel(const ForceArgs a) {
    static_assert(G >= 1 && G <= 4, "1 .. 4 packed groups");
    constexpr int K = 2 * G, WJ = 8, TJ = 256, kBatchTile = 64 * G;
    constexpr int RING_BYTES = STAGES * TJ * 16;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* rings = smem_raw;                                   // [WJ][STAGES][TJ] float4
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + WJ * RING_BYTES);   // full[WJ][STAGES]

    if ((int)blockIdx.x >= a.tile_start[a.n_batch]) return;            // the grid is an upper bound
    const int b = a.cta_batch[blockIdx.x];
    const int i_lo = a.i_off[b] + ((int)blockIdx.x - a.tile_start[b]) * kBatchTile;
    const int i_hi = a.i_off[b + 1];
    const int jr_lo = a.j_off[b], jr_n = a.j_off[b + 1] - jr_lo;
    const int kg = (min(kBatchTile, i_hi - i_lo) + 63) >> 6;           // packed groups that hold particles (1..G)

    const int wj = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t ring = smem_u32(rings + wj * RING_BYTES);
    const uint32_t full0 = smem_u32(bars + wj * STAGES);
    if (lane == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(full0 + 8 * s, 1);
        mbar_fence_init();
    }

    const int j_begin = jr_lo + (int)((long long)jr_n * wj / WJ);
    const int j_end = jr_lo + (int)((long long)jr_n * (wj + 1) / WJ);
    const int n_sub = j_end - j_begin;
    const int n_tiles = (n_sub + TJ - 1) / TJ;
    const unsigned char* src = reinterpret_cast<const unsigned char*>(a.jp + (INDEXED ? 0 : j_begin));
    // INDEXED: indices of the tile that will be issued next (8 per lane), and the issue of one tile's gathers
    int nxt[8];
    auto load_indices = [&](int t) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int e = t * TJ + q * 32 + lane;
            nxt[q] = (t < n_tiles && e < n_sub) ? a.j_index[j_begin + e] : -1;
        }
    };
    auto issue_gather = [&](int t) {                                   // tile t into slot t % STAGES, from the indices in nxt[]
        const uint32_t dst = ring + (t % STAGES) * TJ * 16;
#pragma unroll
        for (int q = 0; q < 8; ++q)
            if (nxt[q] >= 0) cp_async_16(dst + (q * 32 + lane) * 16, a.jp + nxt[q]);
        cp_async_commit();
    };

    const int i_base = i_lo + lane;
    u64 nxi[G], nyi[G], nzi[G];
#pragma unroll
    for (int k2 = 0; k2 < G; ++k2) {
        const int i0 = min(i_base + (2 * k2) * 32, i_hi - 1);
        const int i1 = min(i_base + (2 * k2 + 1) * 32, i_hi - 1);
        nxi[k2] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 0]), neg_canon(a.x_i[3 * (size_t)i1 + 0]));
        nyi[k2] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 1]), neg_canon(a.x_i[3 * (size_t)i1 + 1]));
        nzi[k2] = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 2]), neg_canon(a.x_i[3 * (size_t)i1 + 2]));
    }
    const u64 eps2_2 = pack2(a.eps2, a.eps2);
    const bool half = (G == 1) && (i_hi - i_lo <= 32);                 // ragged tail tile: pack over j (half_sweep)
    u64 hx = 0ull, hy = 0ull, hz = 0ull;
    if (half) {
        const int i0 = min(i_base, i_hi - 1);
        hx = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 0]), neg_canon(a.x_i[3 * (size_t)i0 + 0]));
        hy = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 1]), neg_canon(a.x_i[3 * (size_t)i0 + 1]));
        hz = pack2(neg_canon(a.x_i[3 * (size_t)i0 + 2]), neg_canon(a.x_i[3 * (size_t)i0 + 2]));
    }
    // bounding box of the tile's i-particles (every warp holds the same ones; NaN coordinates drop out of min / max
    // and never coincide with anything)
    float bx0 = __int_as_float(0x7f800000), by0 = bx0, bz0 = bx0, bx1 = -bx0, by1 = -bx0, bz1 = -bx0;
    if (MASKED) {
#pragma unroll
        for (int k2 = 0; k2 < G; ++k2) {
            float lo, hi;
            unpack2(nxi[k2], lo, hi); bx0 = fminf(bx0, fminf(-lo, -hi)); bx1 = fmaxf(bx1, fmaxf(-lo, -hi));
            unpack2(nyi[k2], lo, hi); by0 = fminf(by0, fminf(-lo, -hi)); by1 = fmaxf(by1, fmaxf(-lo, -hi));
            unpack2(nzi[k2], lo, hi); bz0 = fminf(bz0, fminf(-lo, -hi)); bz1 = fmaxf(bz1, fmaxf(-lo, -hi));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            bx0 = fminf(bx0, __shfl_xor_sync(0xffffffffu, bx0, o)); bx1 = fmaxf(bx1, __shfl_xor_sync(0xffffffffu, bx1, o));
            by0 = fminf(by0, __shfl_xor_sync(0xffffffffu, by0, o)); by1 = fmaxf(by1, __shfl_xor_sync(0xffffffffu, by1, o));
            bz0 = fminf(bz0, __shfl_xor_sync(0xffffffffu, bz0, o)); bz1 = fmaxf(bz1, __shfl_xor_sync(0xffffffffu, bz1, o));
        }
        // a subnormal coordinate counts as zero in the loop (add.ftz): widen the box by the smallest normal number
        const float tiny = 1.17549435e-38f;
        bx0 -= tiny; by0 -= tiny; bz0 -= tiny; bx1 += tiny; by1 += tiny; bz1 += tiny;
    }
    __syncthreads();                                                   // barriers initialised

    if (INDEXED) {
        load_indices(0);
        for (int t = 0; t < STAGES; ++t) {                             // STAGES groups in flight, empty beyond the list
            issue_gather(t);
            load_indices(t + 1);
        }
    }
    // each warp is its own producer; a ring slot is refilled by the warp that has just finished reading it
    if (!INDEXED && lane == 0) {
        const int pre = n_tiles < STAGES ? n_tiles : STAGES;
        for (int t = 0; t < pre; ++t) {
            const uint32_t bytes = (uint32_t)min(TJ, n_sub - t * TJ) * 16u;
            mbar_expect_tx(full0 + 8 * t, bytes);
            tma_load_1d(ring + t * TJ * 16, src + (size_t)t * TJ * 16, bytes, full0 + 8 * t);
        }
    }

    double run[K][4];
#pragma unroll
    for (int k = 0; k < K; ++k) { run[k][0] = run[k][1] = run[k][2] = run[k][3] = 0.0; }

    for (int t = 0; t < n_tiles; ++t) {
        const int slot = t % STAGES;
        if (INDEXED) {
            cp_async_wait<STAGES - 1>();                               // this lane's copies of tile t have landed ...
            __syncwarp();                                              // ... and so have the other lanes'
        } else {
            mbar_wait(full0 + 8 * slot, (uint32_t)(t / STAGES) & 1u);
        }
        const int nc = min(TJ, n_sub - t * TJ);                        // TJ == SUB: one Eq. (2) block per tile
        const float4* sp = reinterpret_cast<const float4*>(rings + wj * RING_BYTES + slot * TJ * 16);
        u64 pax[G], pay[G], paz[G], pph[G];
#pragma unroll
        for (int k = 0; k < G; ++k) { pax[k] = 0ull; pay[k] = 0ull; paz[k] = 0ull; pph[k] = 0ull; }
        if (MASKED) {
            // kBatchSub j at a time: a part with no j inside the bounding box of the tile's i-particles cannot hold
            // a coincident pair and runs the untested loop (bit for bit what the masked loop gives there)
            for (int c = 0; c < nc; c += kBatchSub) {
                const int ncc = min(kBatchSub, nc - c);
                bool inside = false;
#pragma unroll
                for (int q = 0; q < kBatchSub; q += 32) {
                    if (q + lane < ncc) {
                        const float4 J = sp[c + q + lane];
                        inside |= (J.x >= bx0) & (J.x <= bx1) & (J.y >= by0) & (J.y <= by1) & (J.z >= bz0) & (J.z <= bz1);
                    }
                }
                if (__any_sync(0xffffffffu, inside)) {
                    if (half) half_sweep<MASK_EXACT, true>(sp + c, ncc, hx, hy, hz, eps2_2, pax[0], pay[0], paz[0], pph[0]);
                    else sweep_dyn<MASK_EXACT, true, G>(kg, sp + c, ncc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
                } else {
                    if (half) half_sweep<MASK_NONE, true>(sp + c, ncc, hx, hy, hz, eps2_2, pax[0], pay[0], paz[0], pph[0]);
                    else sweep_dyn<MASK_NONE, true, G>(kg, sp + c, ncc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
                }
            }
        } else {
            if (half) half_sweep<MASK_NONE, false>(sp, nc, hx, hy, hz, eps2_2, pax[0], pay[0], paz[0], pph[0]);
            else sweep_dyn<MASK_NONE, false, G>(kg, sp, nc, nxi, nyi, nzi, eps2_2, pax, pay, paz, pph);
        }
        if (half) {
            float lo, hi;                                              // both halves belong to particle slot 0
            unpack2(pax[0], lo, hi); run[0][0] += (double)lo + (double)hi;
            unpack2(pay[0], lo, hi); run[0][1] += (double)lo + (double)hi;
            unpack2(paz[0], lo, hi); run[0][2] += (double)lo + (double)hi;
            unpack2(pph[0], lo, hi); run[0][3] += (double)lo + (double)hi;
        } else {
            add_partials<G>(run, pax, pay, paz, pph);
        }
        __syncwarp();                                                  // every lane is done with the slot
        if (INDEXED) {
            issue_gather(t + STAGES);                                  // nxt[] holds tile t + STAGES (or nothing: an empty group)
            load_indices(t + STAGES + 1);
        }
        if (!INDEXED && lane == 0 && t + STAGES < n_tiles) {
            const int tn = t + STAGES;
            const uint32_t bytes = (uint32_t)min(TJ, n_sub - tn * TJ) * 16u;
            mbar_expect_tx(full0 + 8 * slot, bytes);
            tma_load_1d(ring + slot * TJ * 16, src + (size_t)tn * TJ * 16, bytes, full0 + 8 * slot);
        }
    }

    __syncthreads();                                                   // main loops done: the rings are free

    // fixed-order sum over the 8 warps through shared memory (the rings are free)
    double* red = reinterpret_cast<double*>(smem_raw);                 // [WJ][K][4][32]
#pragma unroll
    for (int k = 0; k < K; ++k)
#pragma unroll
        for (int c = 0; c < 4; ++c) red[((wj * K + k) * 4 + c) * 32 + lane] = run[k][c];
    __syncthreads();
    // warp w finishes particle slot k = w (K <= 8 slots, 8 warps)
    if (wj < K) {
        const int k = wj;
        const int i = i_base + k * 32;
        if (i < i_hi) {
            double s[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                s[c] = red[((0 * K + k) * 4 + c) * 32 + lane];
#pragma unroll
                for (int w = 1; w < WJ; ++w) s[c] += red[((w * K + k) * 4 + c) * 32 + lane];
            }
            a.acc[3 * (size_t)i + 0] = (float)s[0];
            a.acc[3 * (size_t)i + 1] = (float)s[1];
            a.acc[3 * (size_t)i + 2] = (float)s[2];
            if (a.pot) a.pot[i] = -(float)s[3];
        }
    }
}

}  // namespace nb
