// nb_small_hermite.cuh -- force + jerk + potential (row f1, Fig. A.4) for SMALL i-sets: the block steps
// of an individual-time-step Hermite integration (BASELINE.json configs[2]: a few hundred to a few thousand
// active particles against everybody) and nb_force_jerk / nb_hermite4 at small N.
//
// The same design as nb_small_kernel (nb_small.cuh), with the Hermite pair arithmetic (nb_hermite_pair.cuh):
//   * PACKED OVER j: the halves of an f32x2 register are two consecutive j-particles, the i-particle (position and velocity)
//     is the broadcast operand; ONE i-particle per thread, 10 packed accumulators (a, J1, J2, phi);
//   * the CTA interleaves its j-chunk into shared memory as pairs -- (x0 x1 y0 y1) (z0 z1 m0 m1) (vx0 vx1 vy0 vy1)
//     (vz0 vz1 - -): four LDS.128 per j-pair, no register shuffling in the loop -- from the packed 32-byte records
//     (x y z m | vx vy vz 0) that the predictor of a Hermite step has written, or from x_j, v_j, m_j directly (nb_force_jerk:
//     no pack launch);
//   * lanes LI x LJ, warps WI x WJ, S j-chunks over CTAs; the partial sums are combined in a FIXED order at every level:
//     shuffles (LJ), shared memory (WJ), distributed shared memory inside a cluster of 2, 4 or 8 CTAs, and -- when S > the
//     cluster size -- FP64 partials in global memory summed by the last-arriving CTA of every (i-tile, slice).  No
//     floating-point atomics: bitwise reproducible, invariant under permutation of the i-set.
//   * every pair is masked (reading R1: all three POSITION differences exactly zero -> the pair adds nothing): an unmasked
//     coincident pair with another velocity would add m dv / eps^3 to the jerk, so there is no speculative form.
// Per pair 27 FP32-pipe instructions (26 without phi) + 1 MUFU; Eq. (2): FP32 partial sums over at most 64
// consecutive j of a slot, FP64 running totals.  jerk = J1 - 3 J2 once, in FP64, in the epilogue.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nb_packed.cuh"
#include "nb_hermite_pair.cuh"
#include "nb_small.cuh"

namespace nb {

struct SmallHermiteArgs {
    const float* x_i;      // [n_i][3]
    const float* v_i;      // [n_i][3]
    const float4* jp;      // [n_j][2] packed records (x y z m | vx vy vz 0), or nullptr: the three arrays below
    const float* xj_raw;   // [n_j][3]
    const float* vj_raw;   // [n_j][3]
    const float* mj_raw;   // [n_j]
    float* acc;            // [n_i][3]
    float* jerk;           // [n_i][3]
    float* pot;            // [n_i] or nullptr
    double* partial;       // [n_i][S / CS][10] when S > CS
    int* tickets;          // [tiles_i * CS] zero between calls, when S > CS
    int n_i;
    int n_j;
    int S;                 // j-chunks across CTAs (grid.y), a multiple of the cluster size
    float eps2;
};

constexpr int kSmallHRoundJ = 2048;      // j-particles staged in shared memory at a time (64 KB + padding)
constexpr int kSmallHBlockPairs = 32;    // Eq. (2): FP32 partial sums over at most 32 j-pairs = 64 j of a slot
constexpr int kSmallHLoadBatch = 2;      // j-pairs (64 B each) a thread loads before it stores them to shared memory
#ifndef NB_SMALL_H_UNROLL
#define NB_SMALL_H_UNROLL 4
#endif
constexpr int kSmallHUnroll = NB_SMALL_H_UNROLL;   // j-pairs per loop iteration (512 x 65536: 54.7 / 50.6 / 52.0 / 49.4 us with 1 / 2 / 3 / 4)

// float4 per j-slot: four per pair, plus one so that the LJ lane groups of a warp (same pair index, LJ different slots)
// read different banks
__host__ __device__ inline int small_h_slot_stride(int slot_len) { return 4 * (slot_len / 2) + 1; }

__device__ __forceinline__ double cluster_ld_double(uint32_t addr) {
    double v;
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}

// NW warps = WI x WJ, lanes = LI x LJ, one i-particle per thread: i-tile = WI * LI.  CS = 1: no cluster; CS = 8: launched in
// clusters of 2, 4 or 8 CTAs along grid.y (the size is read from the hardware).
template <int NW, int LJ, int WJ, bool PHI, int CS>
__global__ void __launch_bounds__(32 * NW) nb_small_hermite_kernel(const SmallHermiteArgs a) {
    constexpr int WI = NW / WJ, LI = 32 / LJ, Q = WJ * LJ, TILE_I = WI * LI, kThreads = 32 * NW, NA = kHermiteAcc;
    static_assert(WI * WJ == NW && LI * LJ == 32, "NW warps of 32 lanes");
    static_assert(TILE_I % CS == 0, "every CTA of a cluster sums a whole slice of the i-tile");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // programmatic dependent launch, as nb_small_kernel: nothing of the previous kernel's output is touched before this
    asm volatile("griddepcontrol.wait;" ::: "memory");

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wi = warp % WI, wj = warp / WI;
    const int li = lane % LI, lj = lane / LI;
    const int q = wj * LJ + lj;                                        // this thread's j-slot
    const int tile0 = blockIdx.x * TILE_I;

    // the i-particle of this thread (clamped load; stores are guarded): -x_i (zeros canonicalised, nb_packed.cuh), -v_i
    u64 ni[6];
    {
        const int i = min(tile0 + wi * LI + li, a.n_i - 1);
        const float x = neg_canon(a.x_i[3 * (size_t)i + 0]), y = neg_canon(a.x_i[3 * (size_t)i + 1]),
                    z = neg_canon(a.x_i[3 * (size_t)i + 2]);
        const float vx = -a.v_i[3 * (size_t)i + 0], vy = -a.v_i[3 * (size_t)i + 1], vz = -a.v_i[3 * (size_t)i + 2];
        ni[0] = pack2(x, x); ni[1] = pack2(y, y); ni[2] = pack2(z, z);
        ni[3] = pack2(vx, vx); ni[4] = pack2(vy, vy); ni[5] = pack2(vz, vz);
    }
    const u64 eps2_2 = pack2(a.eps2, a.eps2);

    double run[NA];                                                    // running totals (outer level of Eq. (2))
#pragma unroll
    for (int c = 0; c < NA; ++c) run[c] = 0.0;

    // the CTA's j-chunk (even boundaries: a j-pair never straddles two CTAs), staged in rounds of at most kSmallHRoundJ
    const int c_lo = (blockIdx.y == 0) ? 0 : ((int)((long long)a.n_j * blockIdx.y / a.S) & ~1);
    const int c_hi = ((int)blockIdx.y + 1 == a.S) ? a.n_j : ((int)((long long)a.n_j * (blockIdx.y + 1) / a.S) & ~1);
    const int chunk_max = (a.n_j + a.S - 1) / a.S + 2;
    const int round_max = min(kSmallHRoundJ, chunk_max);
    const int slot_len = small_slot_len(round_max, Q);
    const int sstride = small_h_slot_stride(slot_len);
    float4* sj = reinterpret_cast<float4*>(smem_raw);                  // [Q][sstride]: 4 float4 per pair

    for (int r_lo = c_lo; r_lo < c_hi; r_lo += kSmallHRoundJ) {
        const int nr = min(kSmallHRoundJ, c_hi - r_lo);
        if (r_lo != c_lo) __syncthreads();                             // the previous round has been consumed
        // staging: one thread per j-pair, kSmallHLoadBatch pairs' loads in flight together
        const int n_pairs_round = (nr + 1) >> 1;
        for (int p0 = threadIdx.x; p0 < n_pairs_round; p0 += kThreads * kSmallHLoadBatch) {
            float4 P0[kSmallHLoadBatch], V0[kSmallHLoadBatch], P1[kSmallHLoadBatch], V1[kSmallHLoadBatch];
#pragma unroll
            for (int u = 0; u < kSmallHLoadBatch; ++u) {
                const int pp = p0 + u * kThreads;
                if (pp >= n_pairs_round) break;
                const size_t j = (size_t)r_lo + 2 * (size_t)pp;
                const bool two = 2 * pp + 1 < nr;                      // false: the round's last pair holds one particle
                if (a.jp) {
                    P0[u] = a.jp[2 * j]; V0[u] = a.jp[2 * j + 1];
                    // an odd count: the second half is a copy with zero mass (adds nothing)
                    P1[u] = two ? a.jp[2 * j + 2] : make_float4(P0[u].x, P0[u].y, P0[u].z, 0.0f);
                    V1[u] = two ? a.jp[2 * j + 3] : V0[u];
                } else {                                               // rows a1 + a2 in one step: no pack launch (nb_force_jerk)
                    const float* xr = a.xj_raw + 3 * j;
                    const float* vr = a.vj_raw + 3 * j;
                    P0[u] = make_float4(xr[0], xr[1], xr[2], a.mj_raw[j]);
                    V0[u] = make_float4(vr[0], vr[1], vr[2], 0.0f);
                    P1[u] = two ? make_float4(xr[3], xr[4], xr[5], a.mj_raw[j + 1]) : make_float4(P0[u].x, P0[u].y, P0[u].z, 0.0f);
                    V1[u] = two ? make_float4(vr[3], vr[4], vr[5], 0.0f) : V0[u];
                }
            }
#pragma unroll
            for (int u = 0; u < kSmallHLoadBatch; ++u) {
                const int pp = p0 + u * kThreads;
                if (pp >= n_pairs_round) break;
                const int jj = 2 * pp, sq = jj / slot_len, pos = jj - sq * slot_len;
                float4* d = sj + (size_t)sq * sstride + 4 * (pos >> 1);
                d[0] = make_float4(P0[u].x, P1[u].x, P0[u].y, P1[u].y);
                d[1] = make_float4(P0[u].z, P1[u].z, P0[u].w, P1[u].w);
                d[2] = make_float4(V0[u].x, V1[u].x, V0[u].y, V1[u].y);
                d[3] = make_float4(V0[u].z, V1[u].z, 0.0f, 0.0f);
            }
        }
        __syncthreads();

        const int len_q = max(0, min(slot_len, nr - q * slot_len));
        const int npairs = (len_q + 1) >> 1;
        const float4* sp = sj + (size_t)q * sstride;
        // Eq. (2) blocks: FP32 partial sums over at most kSmallHBlockPairs pairs, then added to the running totals
        for (int b = 0; b < npairs; b += kSmallHBlockPairs) {
            const int nb_ = min(kSmallHBlockPairs, npairs - b);
            u64 part[NA];
#pragma unroll
            for (int c = 0; c < NA; ++c) part[c] = 0ull;
#pragma unroll kSmallHUnroll
            for (int p = 0; p < nb_; ++p) {
                const float4 A = sp[4 * (b + p)], B = sp[4 * (b + p) + 1], C = sp[4 * (b + p) + 2], D = sp[4 * (b + p) + 3];
                hermite_pair<true, PHI>(pack2(A.x, A.y), pack2(A.z, A.w), pack2(B.x, B.y), pack2(B.z, B.w),
                                        pack2(C.x, C.y), pack2(C.z, C.w), pack2(D.x, D.y),
                                        ni[0], ni[1], ni[2], ni[3], ni[4], ni[5], eps2_2, part);
            }
#pragma unroll
            for (int c = 0; c < NA; ++c) {                             // even-j half first, then odd-j half
                if (!PHI && c == NA - 1) continue;
                float lo, hi;
                unpack2(part[c], lo, hi);
                run[c] += (double)lo;
                run[c] += (double)hi;
            }
        }
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");    // the pair loop is done

    // level 1: the LJ lanes that hold the same i-particle, in the order lj = 0 .. LJ-1 (every lane forms the same sum)
    if (LJ > 1) {
#pragma unroll
        for (int c = 0; c < NA; ++c) {
            const double v = run[c];
            double s = __shfl_sync(0xffffffffu, v, li);
#pragma unroll
            for (int t = 1; t < LJ; ++t) s += __shfl_sync(0xffffffffu, v, li + t * LI);
            run[c] = s;
        }
    }

    // level 2: the WJ warps that hold the same i-particles, through shared memory, in the order wj = 0 .. WJ-1
    __syncthreads();                                                   // the staged j-particles are dead: reuse the memory
    double* red = reinterpret_cast<double*>(smem_raw);                 // [WJ][TILE_I][NA]   (WJ > 1 only)
    double* tile_sum = red + (WJ > 1 ? WJ * TILE_I * NA : 0);          // [TILE_I][NA]
    double* fin = tile_sum + TILE_I * NA;                              // [TILE_I][NA]: the sums the epilogue stores
    if (lj == 0) {
        const int il = wi * LI + li;
        double* dst = (WJ > 1 ? red + ((size_t)wj * TILE_I + il) * NA : tile_sum + (size_t)il * NA);
#pragma unroll
        for (int c = 0; c < NA; ++c) dst[c] = run[c];
    }
    if (WJ > 1) {
        __syncthreads();
        for (int t = threadIdx.x; t < TILE_I * NA; t += kThreads) {
            double s = red[t];
#pragma unroll
            for (int w = 1; w < WJ; ++w) s += red[(size_t)w * TILE_I * NA + t];
            tile_sum[t] = s;
        }
    }

    // level 3: the CTAs of the cluster (consecutive j-chunks of the same i-tile), through distributed shared memory: CTA r
    // sums slice r of the tile over the cluster's CTAs in rank order
    const int cs = (CS > 1) ? (int)cluster_nctarank() : 1;
    const int SLICE = TILE_I / cs;
    const uint32_t rank = (CS > 1) ? cluster_ctarank() : 0u;
    if (CS > 1) cluster_sync_all(); else __syncthreads();
    const int n_groups = a.S / cs;                                     // cluster partials per i-tile
    const int group = blockIdx.y / cs;
    for (int t = threadIdx.x; t < SLICE * NA; t += kThreads) {
        const int e = (int)rank * SLICE * NA + t;                      // element of the tile: (il, c) = (e / NA, e % NA)
        double s;
        if (CS > 1) {
            const uint32_t local = smem_u32(tile_sum + e);
            double v[CS];
#pragma unroll
            for (int c = 0; c < CS; ++c) v[c] = (c < cs) ? cluster_ld_double(cluster_map_shared(local, c)) : 0.0;
            s = v[0];
#pragma unroll
            for (int c = 1; c < CS; ++c)
                if (c < cs) s += v[c];
        } else {
            s = tile_sum[e];
        }
        const int i = tile0 + e / NA;
        if (n_groups == 1) fin[e] = s;
        else if (i < a.n_i) a.partial[((size_t)i * n_groups + group) * NA + (e % NA)] = s;   // a particle's partials are contiguous
    }
    if (CS > 1) cluster_sync_all();                                    // nobody leaves while its shared memory is being read

    // level 4 (S > cluster size): the CTA that arrives LAST at the ticket of its (i-tile, slice) sums the cluster partials in
    // the order group = 0 .. n_groups-1 and leaves the ticket at zero for the next call.  Release / acquire through ONE
    // thread, between two barriers (nb_small.cuh).
    if (n_groups > 1) {
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
        if (!s_last) return;
        for (int t = threadIdx.x; t < SLICE * NA; t += kThreads) {
            const int e = (int)rank * SLICE * NA + t;
            const int i = tile0 + e / NA;
            if (i >= a.n_i) continue;
            const double* p = a.partial + (size_t)i * n_groups * NA + (e % NA);
            double sum = __ldcg(p);
#pragma unroll 8
            for (int g = 1; g < n_groups; ++g) sum += __ldcg(p + (size_t)g * NA);
            fin[e] = sum;
        }
    }
    __syncthreads();

    // epilogue: a, jerk = J1 - 3 J2, phi with its sign
    for (int t = threadIdx.x; t < SLICE * 7; t += kThreads) {
        const int il = (int)rank * SLICE + t / 7, o = t % 7;
        const int i = tile0 + il;
        if (i >= a.n_i) continue;
        const double* s = fin + (size_t)il * NA;
        if (o < 3) a.acc[3 * (size_t)i + o] = (float)s[o];
        else if (o < 6) a.jerk[3 * (size_t)i + (o - 3)] = (float)(s[o] - 3.0 * s[o + 3]);
        else if (a.pot) a.pot[i] = -(float)s[9];
    }
}

}  // namespace nb
