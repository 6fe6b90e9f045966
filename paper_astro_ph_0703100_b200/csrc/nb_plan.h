// nb_plan.h -- launch planner: picks the (i-tile x j-chunk) decomposition of one force call.
//
// Host-only, no CUDA calls, a pure function of (n_i, n_j, sm_count) so that results are
// reproducible (include/nbody_b200.h: "bitwise reproducible ... the planner is a pure function").
//
// Why a planner at all: the paper's scheme keeps one i-particle per
// (virtual) pipeline and sweeps all i for each J-BAG; on a B200 there are
// 148 SMs x 4 schedulers to fill, and n_i / (i per thread) threads alone do not fill them below
// n_i ~ 10^6.  So the j-range is additionally split (a) across the warps of a CTA (WJ) and
// (b) across CTAs (S), and the partial sums are combined in a fixed order.
#pragma once
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <cstdio>

namespace nb {

constexpr int kWarpsPerCta = 8;        // every force CTA has 8 warps = WI * WJ
constexpr int kMaxS = 2048;
// Second pass over the S chunk partials of an i-tile: done inside the force kernel by the tile's last CTA when
// the tile's partials are small (one launch fewer: C0 31 -> 24 us, C2 65 -> 38 us per call), else by a separate
// nb_reduce_kernel launch (a 2048-particle tile with S = 18..30 would keep one CTA busy for ~10 us at the tail).
// Measured per tile: 96 / 144 KB of partials: fused 1.4 / 3.2 us faster; 288 KB: tie; 512 / 576 KB: separate 3 .. 10 us
// faster; 786 / 917 KB / 1.2 MB: separate 8 .. 15 us faster.
constexpr int64_t kFusedReduceBytes = 327680;
inline bool fused_second_pass(int tile_i, int S, double partial_bytes = 32.0) {
    return S > 1 && (double)tile_i * S * partial_bytes <= (double)kFusedReduceBytes;
}

struct Plan {
    int K;            // i-particles per thread (2, 4 or 8; held as K/2 packed pairs)
    int WI;           // warps per CTA along i
    int WJ;           // warps per CTA along j (WI * WJ == 8)
    int S;            // j-chunks across CTAs (grid.y); S > 1 needs the second-pass reduce
    int tiles_i;      // grid.x
    int tile_i;       // i-particles per CTA = 32 * K * WI
    int tile_j;       // j-particles per shared-memory stage
    int stages;       // ring depth
};

inline void ring_shape(int WJ, int* tile_j, int* stages) {
    // shared memory: WJ rings x stages x tile_j x 16 B
    switch (WJ) {
        case 1: *tile_j = 512; *stages = 4; break;   //  32 KB
        case 2: *tile_j = 512; *stages = 4; break;   //  64 KB
        case 4: *tile_j = 256; *stages = 4; break;   //  64 KB
        default: *tile_j = 256; *stages = 3; break;  //  96 KB (WJ = 8)
    }
}

// Cost model in SM clock cycles.  pair_cycles: 13 FP32-pipe lane-ops per pair over 128 lanes per
// clock per SM at the measured ~84 % pipe efficiency of the K = 8 inner loop (profiles/).
inline double plan_cost(int64_t n_i, int64_t n_j, int sm_count, int K, int WI, int WJ, int S,
                        double pair_inst = 13.0, double partial_bytes = 32.0) {
    const double c_fixed = 6000.0;                    // CTA start + first TMA round trip + epilogue
    const double c_reduce_launch = 6000.0;            // second kernel
    const double pair_cycles = pair_inst / (128.0 * 0.84);
    const int tile_i = 32 * K * WI;
    const int64_t tiles_i = (n_i + tile_i - 1) / tile_i;
    const double ctas = double(tiles_i) * S;
    const double waves = double((int64_t)((ctas + sm_count - 1) / sm_count));
    const double j_per_cta = double(n_j) / S;
    // fewer i-particles per thread: more shared-memory reads and loop overhead per pair
    const double k_pen = (K == 8) ? 1.0 : (K == 4 ? 1.06 : 1.15);
    // measured on B200 at full occupancy (one wave of 148 CTAs, K = 8): WJ = 1 / 2 / 4 / 8 reach
    // 82.8 / 77.9 / 81.7 / 81.6 % of the FP32 roofline
    const double wj_pen = (WJ == 1) ? 1.0 : (WJ == 2 ? 1.06 : 1.014);
    double cta_cycles = c_fixed + double(tile_i) * j_per_cta * pair_cycles * k_pen * wj_pen;
    if (WJ > 1) cta_cycles += 1500.0;                 // cross-warp reduction through shared memory
    double cost = waves * cta_cycles;
    if (S > 1) {
        if (fused_second_pass(tile_i, S, partial_bytes))
            cost += 1500.0 + 200.0 * S;               // the last CTA of a tile walks S partials
        else {                                        // separate launch: the partials are written and read back at ~5 TB/s
                                                      // (~2 GHz), or the latency of S loads in a row
            const double bw = double(n_i) * S * partial_bytes / 1250.0, lat = 200.0 * S;
            cost += c_reduce_launch + (bw > lat ? bw : lat);
        }
    }
    return cost;
}

// k_max: largest K the kernel family is instantiated for; pair_inst: FP32-pipe instructions per pair;
// partial_bytes: bytes per (chunk, i) of the second-pass partials; rec_bytes: bytes per j record.
inline Plan make_plan(int64_t n_i, int64_t n_j, int sm_count, int k_max = 8, double pair_inst = 13.0,
                      double partial_bytes = 32.0) {
    if (sm_count <= 0) sm_count = 148;
    Plan best{};
    double best_cost = -1.0;
    static const int k_opts[3] = {8, 4, 2};
    static const int wj_opts[4] = {1, 2, 4, 8};
    for (int k_idx = 0; k_idx < 3; ++k_idx) {
        const int K = k_opts[k_idx];
        if (K > k_max) continue;
        if (K > 2 && n_i <= 32 * (K / 2)) continue;   // a smaller K already covers all i with one warp
        for (int wj_idx = 0; wj_idx < 4; ++wj_idx) {
            const int WJ = wj_opts[wj_idx];
            const int WI = kWarpsPerCta / WJ;
            int64_t s_max = n_j / (8 * WJ);               // every warp-level sub-range gets >= 8 particles
            if (s_max < 1) s_max = 1;
            if (s_max > kMaxS) s_max = kMaxS;
            for (int S = 1; S <= s_max; ++S) {
                const double c = plan_cost(n_i, n_j, sm_count, K, WI, WJ, S, pair_inst, partial_bytes);
                // strict '<' keeps the first (largest K, smallest WJ, smallest S) among equal costs
                if (best_cost < 0.0 || c < best_cost * (1.0 - 1e-9)) {
                    best_cost = c;
                    best.K = K; best.WI = WI; best.WJ = WJ; best.S = S;
                }
            }
        }
    }
    // debugging aid, not part of the ABI: NB_PLAN="K,WI,WJ,S" overrides the choice
    if (const char* env = std::getenv("NB_PLAN")) {
        int k, wi, wj, s;
        if (std::sscanf(env, "%d,%d,%d,%d", &k, &wi, &wj, &s) == 4 && (k == 2 || k == 4 || k == 8) && k <= k_max &&
            wi * wj == kWarpsPerCta && (wj == 1 || wj == 2 || wj == 4 || wj == 8) && s >= 1 && s <= kMaxS) {
            best.K = k; best.WI = wi; best.WJ = wj; best.S = s;
        }
    }
    best.tile_i = 32 * best.K * best.WI;
    best.tiles_i = (int)((n_i + best.tile_i - 1) / best.tile_i);
    ring_shape(best.WJ, &best.tile_j, &best.stages);
    return best;
}

}  // namespace nb
