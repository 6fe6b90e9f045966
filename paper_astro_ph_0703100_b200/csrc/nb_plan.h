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
#include <cmath>

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
// partial_bytes: bytes per (chunk, i) of the second-pass partials.
//
// make_plan_exhaustive tries every S in 1 .. min(n_j / (8 WJ), 2048) for every (K, WJ): ~20 000 cost evaluations,
// 60 .. 220 us on the host -- more than a small call lasts on the device.  It is kept as the DEFINITION of the choice
// (nb_debug.h: nb_debug_plan_exhaustive; tests/test_abi_host.py holds make_plan to it).  make_plan evaluates the same
// cost only where its minimum over S can lie.  For fixed (K, WJ) and a fixed number of waves w = ceil(tiles_i S / #SM)
// the cost is w (C + A / S) + R(S) with R piecewise linear and increasing (fused second pass below the byte threshold,
// separate launch above): convex on each piece, so the minimum over the piece is at one of its ends or next to the
// stationary point sqrt(w A / slope).  Pieces are visited by increasing w until w C_fixed + A tiles_i / #SM -- a lower
// bound for every later piece -- exceeds the best cost found: a few dozen evaluations per (K, WJ), < 3 us in all.
struct PlanChoice { double cost; int K, WI, WJ, S; };

inline Plan finish_plan(int K, int WI, int WJ, int S, int64_t n_i) {
    Plan p{};
    p.K = K; p.WI = WI; p.WJ = WJ; p.S = S;
    p.tile_i = 32 * K * WI;
    p.tiles_i = (int)((n_i + p.tile_i - 1) / p.tile_i);
    ring_shape(WJ, &p.tile_j, &p.stages);
    return p;
}

inline Plan make_plan_exhaustive(int64_t n_i, int64_t n_j, int sm_count, int k_max = 8, double pair_inst = 13.0,
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
    return finish_plan(best.K, best.WI, best.WJ, best.S, n_i);
}

inline Plan make_plan(int64_t n_i, int64_t n_j, int sm_count, int k_max = 8, double pair_inst = 13.0,
                      double partial_bytes = 32.0) {
    if (sm_count <= 0) sm_count = 148;
    static const int k_opts[3] = {8, 4, 2};
    static const int wj_opts[4] = {1, 2, 4, 8};
    PlanChoice best{-1.0, 0, 0, 0, 0};
    for (int k_idx = 0; k_idx < 3; ++k_idx) {
        const int K = k_opts[k_idx];
        if (K > k_max) continue;
        if (K > 2 && n_i <= 32 * (K / 2)) continue;
        for (int wj_idx = 0; wj_idx < 4; ++wj_idx) {
            const int WJ = wj_opts[wj_idx];
            const int WI = kWarpsPerCta / WJ;
            int64_t s_max = n_j / (8 * WJ);
            if (s_max < 1) s_max = 1;
            if (s_max > kMaxS) s_max = kMaxS;
            const int tile_i = 32 * K * WI;
            const int64_t tiles_i = (n_i + tile_i - 1) / tile_i;
            PlanChoice local{-1.0, K, WI, WJ, 0};                         // best of this (K, WJ): the exhaustive order within it
            auto visit = [&](int64_t S) {
                if (S < 1 || S > s_max) return;
                const double c = plan_cost(n_i, n_j, sm_count, K, WI, WJ, (int)S, pair_inst, partial_bytes);
                if (local.cost < 0.0 || c < local.cost * (1.0 - 1e-9) || (S < local.S && c <= local.cost)) { local.cost = c; local.S = (int)S; }
            };
            // work per CTA wave that does not depend on S: A / S with A = tile_i n_j pair_cycles k_pen wj_pen
            const double A = plan_cost(n_i, n_j, sm_count, K, WI, WJ, 1, pair_inst, partial_bytes) /
                                 double((tiles_i + sm_count - 1) / sm_count) - 6000.0 - (WJ > 1 ? 1500.0 : 0.0);
            const double c_fixed = 6000.0 + (WJ > 1 ? 1500.0 : 0.0);
            const double floor_work = A * double(tiles_i) / double(sm_count);
            const int64_t s_fused = (int64_t)((double)kFusedReduceBytes / ((double)tile_i * partial_bytes));   // largest S with a fused second pass
            const double slope_sep = double(n_i) * partial_bytes / 1250.0 > 200.0 ? double(n_i) * partial_bytes / 1250.0 : 200.0;
            visit(1);
            int64_t w = (tiles_i + sm_count - 1) / sm_count;              // waves at S = 1
            int64_t prev_hi = 0;
            for (;; ++w) {
                int64_t hi = w * sm_count / tiles_i;                      // largest S with at most w waves
                if (hi > s_max) hi = s_max;
                const int64_t lo = prev_hi + 1;
                if (hi >= lo) {
                    visit(lo); visit(hi);
                    if (s_fused >= lo && s_fused <= hi) { visit(s_fused); visit(s_fused + 1 <= hi ? s_fused + 1 : hi); }
                    const double slopes[2] = {200.0, slope_sep};
                    for (int q = 0; q < 2; ++q) {
                        const int64_t st = (int64_t)std::sqrt(double(w) * A / slopes[q]);
                        for (int64_t d = -1; d <= 2; ++d) {
                            const int64_t S = st + d;
                            if (S >= lo && S <= hi) visit(S);
                        }
                    }
                    prev_hi = hi;
                }
                if (hi >= s_max) break;
                const double lower = double(w + 1) * c_fixed + floor_work;   // no S with more waves can cost less
                const double ref = local.cost >= 0.0 ? local.cost : -1.0;
                if (ref >= 0.0 && lower >= ref) break;
            }
            if (local.cost >= 0.0 && (best.cost < 0.0 || local.cost < best.cost * (1.0 - 1e-9))) best = local;
        }
    }
    return finish_plan(best.K, best.WI, best.WJ, best.S, n_i);
}

// ------------------------------------------------------------------------------------------------------------------
// Small i-sets (nb_small.cuh): packed over j, lanes LI x LJ, warps WI x WJ, S j-chunks over CTAs in clusters of CS.
struct SmallPlan {
    int NW;           // warps per CTA (8 or 16)
    int KI;           // i-particles per thread (1 or 2)
    int LJ;           // lanes of a warp along j (1, 2 or 4; > 1 only with KI = 1, NW = 8, WJ = 8)
    int WJ;           // warps of the CTA along j (1, 2, 4, 8 or -- NW = 16 -- 16)
    int S;            // j-chunks across CTAs (grid.y), a multiple of CS
    int CS;           // CTAs per thread-block cluster along grid.y (1, 2, 4 or 8)
    int pdl = 1;      // launch with programmatic stream serialisation (NB_SMALL_PDL=0 switches it off: nb_debug.h)
    int tile_i;       // i-particles per CTA = (NW / WJ) * KI * (32 / LJ)
    int tiles_i;      // grid.x
};

constexpr int kSmallClusterMax = 8;
// Which calls nb_force gives to the small-i-set kernel (per call from a CUDA graph of repeated calls, the planner below
// against nb_force_kernel's plan; profiles/r02_small_calls.md "Planner fit"): everything up to 2^25 pairs with at most
// 4096 i-particles -- 1024 x 1024: 3.8 against 6.7 us, C0: 6.3 against 7.6 us, 4096 x 2048: 8.6 against 11.1 us,
// 2048 x 16384: 23.3 against 24.5 us, 1024 x 32768: 22.7 against 25.3 us; ties at 4096 x 4096, 4096 x 8192 and 8192 x 1024 --
// and up to 2^26 pairs with at most 512 (C2: 23.6 against 25.2 us, 512 x 131072: 42.7 against 43.3 us, 32 x 2 000 000:
// 55 against 78 us).  Beyond that nb_force_kernel's K = 8 tiles win (16384 x 16384: 132 against 151 us).
constexpr int64_t kSmallMaxI = 4096;
constexpr int64_t kSmallNarrowI = 512;
constexpr double kSmallMaxPairsNarrow = 67108864.0;    // 2^26, n_i <= 512
constexpr double kSmallMaxPairs = 33554432.0;          // 2^25, n_i <= 4096
constexpr int64_t kSmallVeryNarrowI = 32;              // a handful of i-particles against a long j-set: nb_force_kernel's pack pass over
constexpr double kSmallMaxPairsVeryNarrow = 536870912.0;   // the j-set costs more than the loop (2^29; 32 x 2^23: 177 against 299 us)
inline bool small_by_default(int64_t n_i, int64_t n_j) {
    const double pairs = (double)n_i * (double)n_j;
    return (n_i <= kSmallNarrowI && pairs <= kSmallMaxPairsNarrow) || (n_i <= kSmallMaxI && pairs <= kSmallMaxPairs) ||
           (n_i <= kSmallVeryNarrowI && pairs <= kSmallMaxPairsVeryNarrow);
}
constexpr int kSmallRoundJPlan = 4096;           // = nb::kSmallRoundJ (nb_small.cuh)

// the instantiated shapes (nb_small_launch.cu)
inline bool small_shape_ok(int NW, int KI, int LJ, int WJ, int CS) {
    if (!(NW == 8 || NW == 16) || !(WJ == 1 || WJ == 2 || WJ == 4 || WJ == 8 || (WJ == 16 && NW == 16)) ||
        !(CS == 1 || CS == 2 || CS == 4 || CS == kSmallClusterMax)) return false;
    const bool wide = LJ == 1 && (KI == 1 || KI == 2);                           // throughput shapes: any NW, WJ
    const bool narrow = KI == 1 && (LJ == 2 || LJ == 4) && NW == 8 && WJ == 8;   // 16 or 8 i-particles per CTA
    if (!wide && !narrow) return false;
    return ((NW / WJ) * KI * (32 / LJ)) % CS == 0;
}

// Loop efficiency (fraction of the 13-instruction FP32 roofline) of the j-packed body, measured with micro-loops on a
// B200 (profiles/r02_microloops.md), by i-particles per thread and resident warps per SM: with the exact mask on
// every pair, and without it (the groups SMALL_FLAG finds no mark in; acceleration-only calls).  The cost model below
// uses constants fitted to whole calls instead; this table is what the kernel's design decisions rest on.
inline double small_loop_eff(int KI, int warps_per_sm, bool masked) {
    static const double eff_m[2][3] = {{0.50, 0.65, 0.69}, {0.62, 0.67, 0.70}};   // KI = 1, 2:  8 / 16 / 32 warps per SM
    static const double eff_p[2][3] = {{0.51, 0.73, 0.82}, {0.69, 0.81, 0.85}};
    const int r = KI == 1 ? 0 : 1, c = warps_per_sm >= 32 ? 2 : (warps_per_sm >= 16 ? 1 : 0);
    return masked ? eff_m[r][c] : eff_p[r][c];
}

// SMALL_FLAG (mark the staged j-pairs that may coincide with an i-particle of the tile, mask only their groups) costs
// ~0.8 us of filter build and tests while staging and makes the loop 10-15 % faster: it pays from ~200 packed groups
// per thread when few of the staged j coincide with the tile (C2: 228 groups, 23.5 against 24.6 us; 2048 x 16384, where every
// tile finds its 128 particles among the j: 24.4 against 23.7 us).
constexpr int kSmallFlagMinGroups = 200;
inline bool small_flag_pays(const SmallPlan& p, int64_t n_j) {
    const int64_t chunk = (n_j + p.S - 1) / p.S, Q = (int64_t)p.WJ * p.LJ;
    return p.LJ == 1 && (((chunk + Q - 1) / Q + 1) / 2) * p.KI >= kSmallFlagMinGroups;
}

// Cycles of one small call under a plan.  The FORM follows the kernel's phases (start, staging rounds, pair loop, warp /
// cluster / global sums, waves); the CONSTANTS are fitted to the per-call times of every plan (~500 per shape) on 24 shapes
// from 1 x 4096 to 2048 x 8192, measured from a CUDA graph of 40 calls on a B200 (profiles/r02_small_calls.md, "Planner
// fit"): the plan the model picks is on average 1 % and at worst 5 % slower than the best measured plan of its shape.
inline double small_plan_cost(int64_t n_i, int64_t n_j, int sm_count, int NW, int KI, int LJ, int WJ, int S, int CS) {
    const int tile_i = (NW / WJ) * KI * (32 / LJ);
    const int64_t tiles_i = (n_i + tile_i - 1) / tile_i;
    const int Q = WJ * LJ;
    const double ctas = double(tiles_i) * S;
    const double per_sm = double((int64_t)((ctas + sm_count - 1) / sm_count));      // CTAs on the busiest SM
    const double max_res = NW == 16 ? 1.0 : 2.0;                                    // registers: 86 (KI = 1) / 122 (KI = 2) per thread
    const double resident = per_sm > max_res ? max_res : per_sm;                    // beyond that they run in waves
    double waves = double((int64_t)((per_sm + resident - 1) / resident));
    // A cluster must sit inside one GPC (16 .. 20 SMs): per resident CTA at most 15 clusters of 8 are active at a time on a
    // B200 (ncu launch__cluster_max_active; 120 of the 148 SMs), ~32 of 4, 74 of 2 -- more clusters run as further waves.
    if (CS > 1) {
        const double cap = (CS == 8 ? 15.0 : (CS == 4 ? 32.0 : 74.0)) * resident * sm_count / 148.0;
        const double cw = double((int64_t)((ctas / CS + cap - 1) / cap));
        if (cw > waves) waves = cw;
    }
    const int64_t chunk = (n_j + S - 1) / S;
    const double pairs_per_thread = double((((chunk + Q - 1) / Q) + 1) / 2);
    const double groups = pairs_per_thread * KI;                                    // packed groups of a thread
    // a scheduler holds NW / 4 warps of every resident CTA; a packed group occupies its FMA pipe for 26 cycles
    static const double eff[2][2] = {{0.50, 0.657}, {0.493, 0.663}};                // KI = 1, 2: 8 / >= 16 warps per SM (fitted)
    double loop = resident * groups * (NW / 4) * 26.0 / eff[KI == 1 ? 0 : 1][NW * resident >= 16 ? 1 : 0];
    if (LJ > 1) loop *= 1.0 + 0.14 * LJ;                                            // LJ distinct addresses per LDS.128
    const double lone = groups * 21.0;                                              // one warp's dependent chains
    if (loop < lone) loop = lone;
    const double rounds = double((chunk + kSmallRoundJPlan - 1) / kSmallRoundJPlan);
    const double staged = double(chunk > kSmallRoundJPlan ? kSmallRoundJPlan : chunk);
    double c = 440.0 + 2600.0 * rounds + staged * resident * 0.42;                  // start, staging latency, L2 -> shared memory
    c += loop + 40.0 * KI * (pairs_per_thread / 64.0 + 1.0);                        // Eq. (2) block ends
    c += (WJ > 1) ? 215.0 + 26.0 * WJ : 2250.0;                                     // warp sums; WJ = 1: tiles of 256 .. 1024 particles
    if (CS > 1) c += 2130.0;                                                        // two cluster barriers + DSMEM sums
    const int n_groups = S / CS;
    if (n_groups > 1) c += 1790.0 + 120.0 * n_groups;                               // partials + ticket; final sums per group
    return c * waves;
}

inline int64_t small_plan_key_i(int64_t n_i) { return (n_i + 7) / 8 * 8; }        // every tile size is a multiple of 8

inline SmallPlan make_small_plan(int64_t n_i_exact, int64_t n_j, int sm_count) {
    if (sm_count <= 0) sm_count = 148;
    // the plan is a function of n_i rounded up to a multiple of 8 (same number of i-tiles for every tile size), so that a
    // block-step run whose active set changes every step finds most of its shapes in the library's plan table
    const int64_t n_i = small_plan_key_i(n_i_exact);
    static const int shapes[6][3] = {{16, 2, 1}, {8, 2, 1}, {16, 1, 1}, {8, 1, 1}, {8, 1, 2}, {8, 1, 4}};   // (NW, KI, LJ)
    static const int wj_opts[5] = {1, 2, 4, 8, 16};
    static const int cs_opts[4] = {1, 2, 4, kSmallClusterMax};
    SmallPlan best{};
    double best_cost = -1.0;
    for (int sh = 0; sh < 6; ++sh) {
        const int NW = shapes[sh][0], KI = shapes[sh][1], LJ = shapes[sh][2];
        for (int w = 0; w < 5; ++w) {
            const int WJ = wj_opts[w];
            if (WJ > NW) continue;
            const int tile_i = (NW / WJ) * KI * (32 / LJ);
            if (tile_i > 8 && (int64_t)tile_i >= 2 * n_i) continue;               // a smaller tile covers all i
            const int64_t tiles_i = (n_i + tile_i - 1) / tile_i;
            const int Q = WJ * LJ;
            for (int ci = 0; ci < 4; ++ci) {
                const int CS = cs_opts[ci];
                if (!small_shape_ok(NW, KI, LJ, WJ, CS)) continue;
                int64_t cand[6];
                int n_cand = 0;
                cand[n_cand++] = CS;
                cand[n_cand++] = 2 * CS;
                for (int m = 1; m <= 2; ++m) {                                      // one or two CTAs per SM, rounded down and up
                    cand[n_cand++] = (int64_t)m * sm_count / tiles_i / CS * CS;
                    cand[n_cand++] = (((int64_t)m * sm_count + tiles_i - 1) / tiles_i + CS - 1) / CS * CS;
                }
                const int64_t s_max = (n_j / (2 * Q) / CS) * CS;                     // every slot gets at least one pair
                for (int q = 0; q < n_cand; ++q) {
                    int64_t S = cand[q];
                    if (S > s_max) S = s_max;
                    if (S < CS) S = CS;
                    if (S > kMaxS) S = kMaxS / CS * CS;
                    cand[q] = S;
                    bool seen = false;
                    for (int r = 0; r < q; ++r) seen = seen || cand[r] == S;
                    if (seen) continue;
                    if (CS == 1 && S > 64) continue;                                // without clusters the last CTA of a tile sums alone
                    const double c = small_plan_cost(n_i, n_j, sm_count, NW, KI, LJ, WJ, (int)S, CS);
                    if (best_cost < 0.0 || c < best_cost * (1.0 - 1e-9)) {
                        best_cost = c;
                        best.NW = NW; best.KI = KI; best.LJ = LJ; best.WJ = WJ; best.S = (int)S; best.CS = CS;
                    }
                }
            }
        }
    }
    best.tile_i = (best.NW / best.WJ) * best.KI * (32 / best.LJ);
    best.tiles_i = (int)((n_i + best.tile_i - 1) / best.tile_i);
    return best;
}

// ------------------------------------------------------------------------------------------------------------------
// The small-i-set force + jerk kernel (nb_small_hermite.cuh): one i-particle per thread, 27 instructions per pair, ten sums.
constexpr int kSmallJerkRoundJPlan = 2048;       // = nb::kSmallHRoundJ (nb_small_hermite.cuh)

// the instantiated shapes (nb_small_hermite_launch.cu)
inline bool small_jerk_shape_ok(int NW, int LJ, int WJ, int CS) {
    if (!(CS == 1 || CS == 2 || CS == 4 || CS == kSmallClusterMax)) return false;
    const bool wide = NW == 16 && LJ == 1 && (WJ == 2 || WJ == 4 || WJ == 8 || WJ == 16);
    const bool narrow = NW == 8 && (LJ == 2 || LJ == 4) && WJ == 8;
    if (!wide && !narrow) return false;
    return ((NW / WJ) * (32 / LJ)) % CS == 0;
}

// Cycles of one call: the form of small_plan_cost with the Hermite body (54 FMA-pipe cycles per packed group), 32-byte
// records and ten FP64 sums per particle; the constants are fitted, as there, to the per-call times of every plan on 24
// shapes (3 100 plans; profiles/r02_small_jerk.md): the pick is 1.3 % on average and 7 % at worst behind the best plan.
inline double small_jerk_plan_cost(int64_t n_i, int64_t n_j, int sm_count, int NW, int LJ, int WJ, int S, int CS) {
    const int tile_i = (NW / WJ) * (32 / LJ);
    const int64_t tiles_i = (n_i + tile_i - 1) / tile_i;
    const int Q = WJ * LJ;
    const double ctas = double(tiles_i) * S;
    const double per_sm = double((int64_t)((ctas + sm_count - 1) / sm_count));
    const double max_res = NW == 16 ? 1.0 : 2.0;                                    // registers: 100 .. 122 per thread
    const double resident = per_sm > max_res ? max_res : per_sm;
    double waves = double((int64_t)((per_sm + resident - 1) / resident));
    if (CS > 1) {                                                                   // clusters active at a time (nb_small.cuh)
        const double cap = (CS == 8 ? 15.0 : (CS == 4 ? 31.5 : 74.0)) * resident * sm_count / 148.0;
        const double cw = double((int64_t)((ctas / CS + cap - 1) / cap));
        if (cw > waves) waves = cw;
    }
    const int64_t chunk = (n_j + S - 1) / S;
    const double groups = double((((chunk + Q - 1) / Q) + 1) / 2);                  // packed groups of a thread
    double loop = resident * groups * (NW / 4) * 54.0 / (NW * resident >= 16 ? 0.657 : 0.606);
    if (LJ > 1) loop *= 1.0 + 0.07 * LJ;
    const double lone = groups * 86.5;                                              // one warp's dependent chains
    if (loop < lone) loop = lone;
    const double rounds = double((chunk + kSmallJerkRoundJPlan - 1) / kSmallJerkRoundJPlan);
    const double staged = double(chunk > kSmallJerkRoundJPlan ? kSmallJerkRoundJPlan : chunk);
    double c = 1970.0 * rounds + staged * resident * 0.685;                         // staging latency, L2 -> shared memory
    c += loop + 400.0 * (groups / 32.0 + 1.0);                                      // Eq. (2) block ends: 20 conversions + 20 DADD
    c += 50.0 + 47.6 * WJ * tile_i / 32.0;                                          // warp sums: ten doubles per particle
    if (CS > 1) c += 2220.0;                                                        // two cluster barriers + DSMEM sums
    const int n_groups = S / CS;
    if (n_groups > 1) c += 3200.0 + n_groups * (25.0 + 2.0 * tile_i / CS);          // partials + ticket; final sums of a slice
    return c * waves;
}

inline SmallPlan make_small_jerk_plan(int64_t n_i_exact, int64_t n_j, int sm_count) {
    if (sm_count <= 0) sm_count = 148;
    static const int shapes[6][3] = {{16, 1, 2}, {16, 1, 4}, {16, 1, 8}, {16, 1, 16}, {8, 2, 8}, {8, 4, 8}};   // (NW, LJ, WJ)
    static const int cs_opts[4] = {1, 2, 4, kSmallClusterMax};
    const int64_t n_i = small_plan_key_i(n_i_exact);
    SmallPlan best{};
    double best_cost = -1.0;
    for (int sh = 0; sh < 6; ++sh) {
        const int NW = shapes[sh][0], LJ = shapes[sh][1], WJ = shapes[sh][2];
        const int tile_i = (NW / WJ) * (32 / LJ);
        if (tile_i > 8 && (int64_t)tile_i >= 2 * n_i) continue;
        const int64_t tiles_i = (n_i + tile_i - 1) / tile_i;
        const int Q = WJ * LJ;
        for (int ci = 0; ci < 4; ++ci) {
            const int CS = cs_opts[ci];
            if (!small_jerk_shape_ok(NW, LJ, WJ, CS)) continue;
            int64_t cand[6];
            int n_cand = 0;
            cand[n_cand++] = CS;
            cand[n_cand++] = 2 * CS;
            for (int m = 1; m <= 2; ++m) {
                cand[n_cand++] = (int64_t)m * sm_count / tiles_i / CS * CS;
                cand[n_cand++] = (((int64_t)m * sm_count + tiles_i - 1) / tiles_i + CS - 1) / CS * CS;
            }
            const int64_t s_max = (n_j / (2 * Q) / CS) * CS;
            for (int q = 0; q < n_cand; ++q) {
                int64_t S = cand[q];
                if (S > s_max) S = s_max;
                if (S < CS) S = CS;
                if (S > kMaxS) S = kMaxS / CS * CS;
                cand[q] = S;
                bool seen = false;
                for (int r = 0; r < q; ++r) seen = seen || cand[r] == S;
                if (seen) continue;
                if (CS == 1 && S > 64) continue;
                const double c = small_jerk_plan_cost(n_i, n_j, sm_count, NW, LJ, WJ, (int)S, CS);
                if (best_cost < 0.0 || c < best_cost * (1.0 - 1e-9)) {
                    best_cost = c;
                    best.NW = NW; best.KI = 1; best.LJ = LJ; best.WJ = WJ; best.S = (int)S; best.CS = CS;
                }
            }
        }
    }
    best.tile_i = (best.NW / best.WJ) * (32 / best.LJ);
    best.tiles_i = (int)((n_i + best.tile_i - 1) / best.tile_i);
    return best;
}

// Which evaluations take it (per call from a CUDA graph, best plan of this kernel against nb_hermite_kernel's;
// profiles/r02_small_jerk.md).
//  * Hermite steps (nb_hermite4, nb_hermite4_block_step), whose predictor has packed the j-records: up to 2^22 pairs (2^23
//    for at most 512 i-particles) --
//    256 x 256: 5.3 against 7.8 us, 100 x 10000: 9.2 against 14.5, 64 x 65536: 15.6 against 26.1, 2048 x 2048: 12.5 against
//    13.4; a tie at 1024 x 4096, and beyond nb_hermite_kernel wins (2048 x 8192: 28.9 against 26.2, 256 x 65536: 31.6 against
//    30.0): ONE i-particle per thread gives the loop no more independent chains than the i-packed K = 2 / 4 body.
//  * nb_force_jerk on x_j, v_j, m_j: this kernel packs while it stages, nb_hermite_kernel needs nb_pack_jv_kernel first, so
//    it stays ahead up to 2^25 pairs (4096 i-particles) and 2^26 pairs (1024): 256 x 256: 3.3 against 7.5 us, 2048 x 2048:
//    9.9 against 13.7, 4096 x 4096: 25.6 against 28.0, 2048 x 16384: 44.1 against 46.7, 1024 x 65536: 82.7 against 87.0;
//    2048 x 65536: 157 against 148.
constexpr int64_t kSmallJerkMaxI = 4096;
constexpr double kSmallJerkMaxPairs = 4194304.0;           // 2^22: records already packed
constexpr int64_t kSmallJerkStepsNarrowI = 512;
constexpr double kSmallJerkMaxPairsNarrow = 8388608.0;     // 2^23: records already packed, n_i <= 512 (block steps: 128 of
                                                           // 65536 active 25.9 against 31.3 us, 512 of 16384 26.0 against 27.1)
constexpr double kSmallJerkMaxPairsRaw = 33554432.0;       // 2^25: nb_force_jerk
constexpr int64_t kSmallJerkNarrowI = 1024;
constexpr double kSmallJerkMaxPairsRawNarrow = 67108864.0; // 2^26: nb_force_jerk, n_i <= 1024
constexpr int64_t kSmallJerkVeryNarrowI = 256;             // ... and 2^28 for n_i <= 256: nb_pack_jv_kernel over a long j-set costs
constexpr double kSmallJerkMaxPairsRawVeryNarrow = 268435456.0;   // more than the loop gains (128 x 2^20: 166 against 202 us)
constexpr double kSmallJerkMaxPairsRawHandful = 536870912.0;      // 2^29 for n_i <= 32 (32 x 2^23: 369 against 653 us)
inline bool small_jerk_by_default(int64_t n_i, int64_t n_j, bool prepacked) {
    const double pairs = (double)n_i * (double)n_j;
    if (n_i > kSmallJerkMaxI) return false;
    if (prepacked) return pairs <= kSmallJerkMaxPairs || (n_i <= kSmallJerkStepsNarrowI && pairs <= kSmallJerkMaxPairsNarrow);
    return pairs <= kSmallJerkMaxPairsRaw || (n_i <= kSmallJerkNarrowI && pairs <= kSmallJerkMaxPairsRawNarrow) ||
           (n_i <= kSmallJerkVeryNarrowI && pairs <= kSmallJerkMaxPairsRawVeryNarrow) ||
           (n_i <= kSmallVeryNarrowI && pairs <= kSmallJerkMaxPairsRawHandful);
}

}  // namespace nb
