// nbody_b200.cu -- C-ABI shim, workspace and launch logic of libnbody_b200.so (include/nbody_b200.h).
#include "../../include/nbody_b200.h"
#include "../../include/nb_debug.h"

#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <tuple>
#include <unordered_map>
#include <utility>
#include <vector>

#include "nb_kernels.cuh"
#include "nb_hermite.cuh"
#include "nb_batched.cuh"
#include "nb_pipelines.cuh"
#include "nb_plan.h"
#include "nb_small.cuh"
#include "nb_small_launch.h"
#include "nb_small_hermite.cuh"
#include "nb_small_hermite_launch.h"

#define NB_VERSION 100

namespace {

thread_local int t_last_cuda_error = 0;
thread_local int64_t t_launches = 0;
thread_local bool t_profile = false;
thread_local std::vector<std::pair<cudaEvent_t, cudaEvent_t>> t_events;

#define NB_CUDA(call)                                  \
    do {                                               \
        cudaError_t e__ = (call);                      \
        if (e__ != cudaSuccess) {                      \
            t_last_cuda_error = (int)e__;              \
            (void)cudaGetLastError();                  \
            return NB_ERR_CUDA;                        \
        }                                              \
    } while (0)

struct DeviceInfo {
    bool known = false;
    bool supported = false;
    int sm_count = 0;
};

struct Workspace {
    void* jp = nullptr;        size_t jp_bytes = 0;        // packed pair records
    void* partial = nullptr;   size_t partial_bytes = 0;   // [S][n_i] double4
    void* stage = nullptr;     size_t stage_bytes = 0;     // device copies for nb_force_host
    void* tickets = nullptr;   size_t tickets_bytes = 0;   // fused second pass: one counter per i-tile, zero between calls
    void* coin = nullptr;      size_t coin_bytes = 0;      // coincidence pre-pass: flag | lists | hash table
    void* tiles = nullptr;     size_t tiles_bytes = 0;     // batched calls: first CTA of every sub-problem
    void* pipe = nullptr;      size_t pipe_bytes = 0;      // generalised kernel: [S][n_i][FDIM] double
    void* hstate = nullptr;    size_t hstate_bytes = 0;    // Hermite integrator: xp, vp, a1, j1
    void* jp2 = nullptr;       size_t jp2_bytes = 0;       // force + jerk: 32-byte j records
    void* hpartial = nullptr;  size_t hpartial_bytes = 0;  // force + jerk: [S][n_i][10] double
    std::recursive_mutex busy;                             // held while a call grows the buffers and enqueues work that uses them
};

// Debugging switches (include/nb_debug.h): read from the environment once, changed only through nb_debug_set.
struct Knobs {
    bool plan_set = false;       int pK = 0, pWI = 0, pWJ = 0, pS = 0;                 // NB_PLAN
    bool small_plan_set = false; int sNW = 0, sKI = 0, sLJ = 0, sWJ = 0, sS = 0, sCS = 0;   // NB_SMALL_PLAN
    int small = -1;              // NB_SMALL: -1 default, 0 never, 1 always
    int small_jerk = -1;         // NB_SMALL_JERK: -1 default, 0 never, 1 always (nb_force_jerk and the block step)
    bool small_jerk_plan_set = false; int jNW = 0, jLJ = 0, jWJ = 0, jS = 0, jCS = 0;   // NB_SMALL_JERK_PLAN
    int small_pdl = -1;          // NB_SMALL_PDL: -1 / 1 programmatic dependent launch of nb_small_kernel, 0 plain launch
    int small_mask = -1;         // NB_SMALL_MASK: -1 default (marked pairs), nb::SMALL_EXACT = every pair masked
    int mask = -1;               // NB_MASK: -1 default, else nb::MODE_*
    int fused = -1;              // NB_FUSED_REDUCE
    int direct = -1;             // NB_DIRECT
    int step_graph = -1;         // NB_STEP_GRAPH
    int hermite_fuse = -1;       // NB_HERMITE_FUSE: 0 = correct and predict as separate launches
    int batch_tile = 0;          // NB_BATCH_TILE
};

std::mutex g_mutex;
std::atomic<const Knobs*> g_knobs{nullptr};
std::atomic<int64_t> g_plans_computed{0};
DeviceInfo g_dev[64];
std::map<std::pair<int, cudaStream_t>, Workspace> g_ws;
std::map<std::tuple<int64_t, int64_t, int>, nb::Plan> g_plans;
std::map<std::tuple<int64_t, int64_t, int>, nb::Plan> g_hplans;
std::map<std::tuple<int64_t, int64_t, int>, nb::SmallPlan> g_splans;
std::map<std::tuple<int64_t, int64_t, int>, nb::SmallPlan> g_sjplans;

// ---- debugging switches
bool parse_knob(Knobs* k, const char* key, const char* value) {
    const bool unset = !value || !value[0];
    if (!std::strcmp(key, "NB_PLAN")) {
        if (unset) { k->plan_set = false; return true; }
        int a, b, c, d;
        if (std::sscanf(value, "%d,%d,%d,%d", &a, &b, &c, &d) != 4) return false;
        if (!((a == 2 || a == 4 || a == 8) && b * c == nb::kWarpsPerCta && (c == 1 || c == 2 || c == 4 || c == 8) && d >= 1 && d <= nb::kMaxS)) return false;
        k->plan_set = true; k->pK = a; k->pWI = b; k->pWJ = c; k->pS = d;
        return true;
    }
    if (!std::strcmp(key, "NB_SMALL_PLAN")) {
        if (unset) { k->small_plan_set = false; return true; }
        int nw, ki, lj, wj, ss, cs;
        if (std::sscanf(value, "%d,%d,%d,%d,%d,%d", &nw, &ki, &lj, &wj, &ss, &cs) != 6) return false;
        if (!(nb::small_shape_ok(nw, ki, lj, wj, cs) && ss >= cs && ss % cs == 0 && ss <= nb::kMaxS)) return false;
        k->small_plan_set = true; k->sNW = nw; k->sKI = ki; k->sLJ = lj; k->sWJ = wj; k->sS = ss; k->sCS = cs;
        return true;
    }
    if (!std::strcmp(key, "NB_SMALL_JERK")) {
        if (unset) { k->small_jerk = -1; return true; }
        if (std::strcmp(value, "0") && std::strcmp(value, "1")) return false;
        k->small_jerk = value[0] - '0';
        return true;
    }
    if (!std::strcmp(key, "NB_SMALL_JERK_PLAN")) {
        if (unset) { k->small_jerk_plan_set = false; return true; }
        int nw, lj, wj, ss, cs;
        if (std::sscanf(value, "%d,%d,%d,%d,%d", &nw, &lj, &wj, &ss, &cs) != 5) return false;
        if (!(nb::small_jerk_shape_ok(nw, lj, wj, cs) && ss >= cs && ss % cs == 0 && ss <= nb::kMaxS)) return false;
        k->small_jerk_plan_set = true; k->jNW = nw; k->jLJ = lj; k->jWJ = wj; k->jS = ss; k->jCS = cs;
        return true;
    }
    if (!std::strcmp(key, "NB_HERMITE_FUSE")) {
        if (unset) { k->hermite_fuse = -1; return true; }
        if (std::strcmp(value, "0") && std::strcmp(value, "1")) return false;
        k->hermite_fuse = value[0] - '0';
        return true;
    }
    if (!std::strcmp(key, "NB_SMALL_PDL")) {
        if (unset) { k->small_pdl = -1; return true; }
        if (std::strcmp(value, "0") && std::strcmp(value, "1")) return false;
        k->small_pdl = value[0] - '0';
        return true;
    }
    if (!std::strcmp(key, "NB_SMALL_MASK")) {
        if (unset) { k->small_mask = -1; return true; }
        if (value[0] == 'e') k->small_mask = nb::SMALL_EXACT; else if (value[0] == 'f') k->small_mask = nb::SMALL_FLAG; else return false;
        return true;
    }
    if (!std::strcmp(key, "NB_MASK")) {
        if (unset) { k->mask = -1; return true; }
        if (value[0] == 'e') k->mask = nb::MODE_EXACT; else if (value[0] == 'b') k->mask = nb::MODE_BLOOM;
        else if (value[0] == 'l') k->mask = nb::MODE_LIST; else return false;
        return true;
    }
    int* flag = !std::strcmp(key, "NB_SMALL") ? &k->small : !std::strcmp(key, "NB_FUSED_REDUCE") ? &k->fused :
                !std::strcmp(key, "NB_DIRECT") ? &k->direct : !std::strcmp(key, "NB_STEP_GRAPH") ? &k->step_graph : nullptr;
    if (flag) {
        if (unset) { *flag = -1; return true; }
        if (value[0] != '0' && value[0] != '1') return false;
        *flag = value[0] - '0';
        return true;
    }
    if (!std::strcmp(key, "NB_BATCH_TILE")) {
        if (unset) { k->batch_tile = 0; return true; }
        const int t = std::atoi(value);
        if (t != 64 && t != 128 && t != 256) return false;
        k->batch_tile = t;
        return true;
    }
    return false;
}

const char* const kKnobKeys[] = {"NB_PLAN", "NB_SMALL_PLAN", "NB_SMALL", "NB_SMALL_MASK", "NB_SMALL_PDL", "NB_SMALL_JERK", "NB_SMALL_JERK_PLAN", "NB_MASK", "NB_FUSED_REDUCE", "NB_DIRECT", "NB_STEP_GRAPH", "NB_HERMITE_FUSE", "NB_BATCH_TILE"};

// the current switches: one atomic load per call; the environment is read once, here
const Knobs& knobs() {
    const Knobs* k = g_knobs.load(std::memory_order_acquire);
    if (k) return *k;
    std::lock_guard<std::mutex> lock(g_mutex);
    k = g_knobs.load(std::memory_order_acquire);
    if (k) return *k;
    Knobs* fresh = new Knobs();
    for (const char* key : kKnobKeys)
        if (const char* v = std::getenv(key)) (void)parse_knob(fresh, key, v);   // a value that does not parse is ignored
    g_knobs.store(fresh, std::memory_order_release);
    return *fresh;
}

// ---- per (device, stream) workspace, locked for the duration of one call's enqueue sequence
struct WsGuard {
    Workspace* ws;
    std::unique_lock<std::recursive_mutex> hold;
    WsGuard(int dev, cudaStream_t stream) {
        {
            std::lock_guard<std::mutex> lock(g_mutex);
            ws = &g_ws[std::make_pair(dev, stream)];
        }
        hold = std::unique_lock<std::recursive_mutex>(ws->busy);
    }
};

void free_workspace(Workspace* w) {
    void** bufs[] = {&w->jp, &w->partial, &w->stage, &w->coin, &w->tickets, &w->jp2, &w->tiles, &w->pipe, &w->hstate, &w->hpartial};
    for (void** b : bufs) {
        if (*b) (void)cudaFree(*b);
        *b = nullptr;
    }
    w->jp_bytes = w->partial_bytes = w->stage_bytes = w->coin_bytes = w->tickets_bytes = w->jp2_bytes = w->tiles_bytes =
        w->pipe_bytes = w->hstate_bytes = w->hpartial_bytes = 0;
}

int device_info(int* dev_out, DeviceInfo* out) {
    int dev = 0;
    NB_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return NB_ERR_UNSUPPORTED_DEVICE;
    std::lock_guard<std::mutex> lock(g_mutex);
    DeviceInfo& d = g_dev[dev];
    if (!d.known) {
        int major = 0;
        NB_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        NB_CUDA(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
        d.supported = (major == 10);
        d.known = true;
    }
    *dev_out = dev;
    *out = d;
    return d.supported ? NB_OK : NB_ERR_UNSUPPORTED_DEVICE;
}

// grow-only, stream-ordered
int ensure(void** ptr, size_t* have, size_t need, cudaStream_t stream) {
    if (need <= *have) return NB_OK;
    size_t want = need + need / 4 + 256;
    void* fresh = nullptr;
    cudaError_t e = cudaMallocAsync(&fresh, want, stream);
    if (e != cudaSuccess) {
        t_last_cuda_error = (int)e;
        (void)cudaGetLastError();
        return NB_ERR_ALLOC;
    }
    if (*ptr) NB_CUDA(cudaFreeAsync(*ptr, stream));
    *ptr = fresh;
    *have = want;
    return NB_OK;
}

constexpr double kHermiteInstPerPair = 27.0;     // force + jerk + potential (row f1): FP32-pipe instructions per pair
constexpr double kHermitePartialBytes = 80.0;    // ... and bytes per (chunk, i) of its second-pass partials

// NB_PLAN (nb_debug.h) overrides the planner's choice; a forced plan is not remembered
bool forced_plan(const Knobs& kn, int k_max, int64_t n_i, nb::Plan* out) {
    if (!kn.plan_set || kn.pK > k_max) return false;
    *out = nb::finish_plan(kn.pK, kn.pWI, kn.pWJ, kn.pS, n_i);
    return true;
}

// The planner costs ~3 us per new shape (nb_plan.h); repeated shapes are served from a small per-process table.
nb::Plan cached_plan(int64_t n_i, int64_t n_j, int sm_count, bool jerk = false) {
    nb::Plan p;
    if (forced_plan(knobs(), jerk ? 4 : 8, n_i, &p)) return p;
    auto& table = jerk ? g_hplans : g_plans;
    const auto key = std::make_tuple(n_i, n_j, sm_count);
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        auto it = table.find(key);
        if (it != table.end()) return it->second;
    }
    p = jerk ? nb::make_plan(n_i, n_j, sm_count, 4, kHermiteInstPerPair, kHermitePartialBytes)
             : nb::make_plan(n_i, n_j, sm_count);                          // outside the lock
    g_plans_computed.fetch_add(1, std::memory_order_relaxed);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (table.size() > 4096) table.clear();
    table[key] = p;
    return p;
}

// Capturing and instantiating the step graph costs ~140 us, a replayed step saves ~2 us: from 64 steps on it pays
// (N = 256 leapfrog: 32 steps 8.7 against 8.2 us per step eagerly, 100 steps 5.7 against 7.3; profiles/r02_small_jerk.md)
constexpr int64_t kStepGraphMinSteps = 64;

// Steps captured into ONE graph by nb_leapfrog_kdk / nb_hermite4 (at most 8; fewer for short runs so that the graph is replayed
// at least four times)
int64_t graph_steps(int64_t remaining) {
    const int64_t u = remaining / 4;
    return u < 1 ? 1 : (u > 8 ? 8 : u);
}

// The default streams (NULL / legacy and per-thread) cannot be captured, and they are what most callers pass.  A long run on a
// small system is then moved to a private non-blocking stream of the device for the duration of the call: the private stream
// first waits for everything enqueued on the caller's stream so far, the caller's stream then waits for the run -- stream order
// as the caller sees it is unchanged, and the step graph becomes possible.  Host threads that detour on the same device are
// serialised for the duration of the enqueue (their work would be serialised on the device anyway).
struct StreamDetour {
    struct PerDevice { cudaStream_t stream = nullptr; cudaEvent_t ev_in = nullptr, ev_out = nullptr; std::mutex busy; };
    static PerDevice& slot(int dev) { static PerDevice table[64]; return table[dev & 63]; }
    PerDevice* pd = nullptr;
    cudaStream_t user = nullptr;
    std::unique_lock<std::mutex> lock;
    // on success *stream is the private stream
    int begin(int dev, cudaStream_t user_stream, cudaStream_t* stream) {
        PerDevice& d = slot(dev);
        lock = std::unique_lock<std::mutex>(d.busy);
        if (!d.stream) {
            NB_CUDA(cudaStreamCreateWithFlags(&d.stream, cudaStreamNonBlocking));
            NB_CUDA(cudaEventCreateWithFlags(&d.ev_in, cudaEventDisableTiming));
            NB_CUDA(cudaEventCreateWithFlags(&d.ev_out, cudaEventDisableTiming));
        }
        NB_CUDA(cudaEventRecord(d.ev_in, user_stream));
        NB_CUDA(cudaStreamWaitEvent(d.stream, d.ev_in, 0));
        pd = &d;
        user = user_stream;
        *stream = d.stream;
        return NB_OK;
    }
    ~StreamDetour() {                                                  // on every way out of the call, errors included
        if (!pd) return;
        if (cudaEventRecord(pd->ev_out, pd->stream) == cudaSuccess) (void)cudaStreamWaitEvent(user, pd->ev_out, 0);
    }
};
// whether nb_leapfrog_kdk / nb_hermite4 would replay their steps from a graph if the stream allowed it
bool wants_step_graph(int64_t n, int64_t n_steps) {
    return n_steps >= kStepGraphMinSteps && n <= 32768 && !t_profile && knobs().step_graph != 0;
}

// the small-i-set kernel's planner scores ~1000 candidate decompositions (~10 us): the same table serves repeated shapes
nb::SmallPlan cached_small_plan(int64_t n_i, int64_t n_j, int sm_count) {
    const auto key = std::make_tuple(nb::small_plan_key_i(n_i), n_j, sm_count);
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        auto it = g_splans.find(key);
        if (it != g_splans.end()) return it->second;
    }
    const nb::SmallPlan p = nb::make_small_plan(n_i, n_j, sm_count);       // outside the lock
    g_plans_computed.fetch_add(1, std::memory_order_relaxed);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (g_splans.size() > 4096) g_splans.clear();
    g_splans[key] = p;
    return p;
}

nb::SmallPlan cached_small_jerk_plan(int64_t n_i, int64_t n_j, int sm_count) {
    const auto key = std::make_tuple(nb::small_plan_key_i(n_i), n_j, sm_count);
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        auto it = g_sjplans.find(key);
        if (it != g_sjplans.end()) return it->second;
    }
    const nb::SmallPlan p = nb::make_small_jerk_plan(n_i, n_j, sm_count);  // outside the lock
    g_plans_computed.fetch_add(1, std::memory_order_relaxed);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (g_sjplans.size() > 4096) g_sjplans.clear();
    g_sjplans[key] = p;
    return p;
}

// An UNMASKED coincident pair must stay finite (m * rsqrt(eps2)^3 = m * 2^60 at the threshold): the list mode and
// the acceleration-only path need eps2 >= 2^-40; below that (and for eps2 == 0) every pair is masked.
constexpr float kUnmaskedMinEps2 = 9.094947017729282e-13f;

// Where the coincident pairs are found (reading R1), by call size:
//   >= 2^32 pairs   MODE_LIST: hash-join pre-pass (three extra O(n) launches, ~35 us), no test in the hot loop;
//   >= 2^25 pairs   MODE_BLOOM: the force kernel tests every 256-j block against a Bloom filter of its warp's
//                   i-positions (~1 % of the loop), no pre-pass -- and the small-call one-launch path stays possible;
//   smaller, eps2 < 2^-40, per-i softening below the list size: MODE_EXACT, every pair masked.
constexpr double kListMinPairs = 4294967296.0;   // 2^32
constexpr double kListMinPairsNoBloom = 536870912.0;   // 2^29 (per-i softening has no Bloom instantiation)
constexpr double kBloomMinPairs = 33554432.0;    // 2^25
constexpr double kListMinPairsJerk = 1073741824.0;   // 2^30: the jerk kernel's pre-pass pays off earlier (measured tie at N = 32768)

int pick_mode(int64_t n_i, int64_t n_j, float eps2, bool bloom_ok, double list_min_pairs = kListMinPairs) {
    // debugging aid (nb_debug.h): NB_MASK forces a mode (bloom and list still need eps2 >= 2^-40, list n_j <= 2^29)
    const int forced = knobs().mask;
    if (forced == nb::MODE_EXACT) return nb::MODE_EXACT;
    if (eps2 < kUnmaskedMinEps2) return nb::MODE_EXACT;
    const bool list_ok = n_j <= ((int64_t)1 << 29);                    // the 32-bit hash table holds 2 n_j <= 2^30 slots
    const double pairs = (double)n_i * (double)n_j;
    if (!bloom_ok) return (list_ok && (forced == nb::MODE_LIST || pairs >= kListMinPairsNoBloom)) ? nb::MODE_LIST : nb::MODE_EXACT;
    if (forced == nb::MODE_LIST) return list_ok ? nb::MODE_LIST : nb::MODE_EXACT;
    if (forced == nb::MODE_BLOOM) return nb::MODE_BLOOM;
    if (list_ok && pairs >= list_min_pairs) return nb::MODE_LIST;
    return pairs >= kBloomMinPairs ? nb::MODE_BLOOM : nb::MODE_EXACT;
}

// One launch of a dominant kernel: raises the kernel's dynamic shared-memory limit once per device, brackets the
// launch with two events on the launching stream while nb_profile_enable is on, counts it.
template <class Kernel, class Args>
int launch_dominant(Kernel kern, std::atomic<uint64_t>* configured, dim3 grid, unsigned threads, size_t smem, cudaStream_t stream,
                    const Args& args) {
    int dev = 0;
    NB_CUDA(cudaGetDevice(&dev));
    const uint64_t bit = 1ull << (dev & 63);                           // bit d: device d has the raised limit (idempotent: a race only repeats the call)
    if (!(configured->load(std::memory_order_acquire) & bit)) {
        NB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured->fetch_or(bit, std::memory_order_release);
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (t_profile) {
        NB_CUDA(cudaEventCreate(&e0));
        NB_CUDA(cudaEventCreate(&e1));
        NB_CUDA(cudaEventRecord(e0, stream));
    }
    kern<<<grid, threads, smem, stream>>>(args);
    NB_CUDA(cudaGetLastError());
    if (t_profile) {
        NB_CUDA(cudaEventRecord(e1, stream));
        t_events.emplace_back(e0, e1);
    }
    ++t_launches;
    return NB_OK;
}

template <int K, int WI, int WJ, int TJ, int STAGES, int MODE, bool EPS_I, bool PHI = true, bool DIRECT = false>
int launch_force_inst(const nb::ForceArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    constexpr size_t ring = (size_t)WJ * STAGES * TJ * 16;
    constexpr size_t red = (WJ > 1) ? (size_t)WJ * K * 4 * (WI * 32) * sizeof(double) : 0;
    constexpr size_t bloom = (MODE == nb::MODE_BLOOM) ? (size_t)WI * nb::kBloomWords * sizeof(uint32_t) : 0;
    constexpr size_t smem = (ring + bloom > red ? ring + bloom : red) + 2 * WJ * STAGES * sizeof(uint64_t) + 128;
    static std::atomic<uint64_t> configured{0};
    return launch_dominant(nb::nb_force_kernel<K, WI, WJ, TJ, STAGES, MODE, EPS_I, PHI, DIRECT>, &configured,
                           dim3((unsigned)plan.tiles_i, (unsigned)plan.S, 1), 32 * WI * WJ, smem, stream, args);
}

// tile_j / stages per WJ must match nb::ring_shape (nb_plan.h)
template <int K, int MODE, bool EPS_I, bool DIRECT = false>
int launch_force_k(const nb::ForceArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    switch (plan.WJ) {
        case 1: return launch_force_inst<K, 8, 1, 512, 4, MODE, EPS_I, true, DIRECT>(args, plan, stream);
        case 2: return launch_force_inst<K, 4, 2, 512, 4, MODE, EPS_I, true, DIRECT>(args, plan, stream);
        case 4: return launch_force_inst<K, 2, 4, 256, 4, MODE, EPS_I, true, DIRECT>(args, plan, stream);
        default: return launch_force_inst<K, 1, 8, 256, 3, MODE, EPS_I, true, DIRECT>(args, plan, stream);
    }
}

// pot_out == NULL on a large call: the 12-instruction loop without the potential (K = 8, list mode only)
int launch_force_nophi(const nb::ForceArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    switch (plan.WJ) {
        case 1: return launch_force_inst<8, 8, 1, 512, 4, nb::MODE_LIST, false, false>(args, plan, stream);
        case 2: return launch_force_inst<8, 4, 2, 512, 4, nb::MODE_LIST, false, false>(args, plan, stream);
        case 4: return launch_force_inst<8, 2, 4, 256, 4, nb::MODE_LIST, false, false>(args, plan, stream);
        default: return launch_force_inst<8, 1, 8, 256, 3, nb::MODE_LIST, false, false>(args, plan, stream);
    }
}

template <int MODE, bool EPS_I = false, bool DIRECT = false>
int launch_force(const nb::ForceArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    switch (plan.K) {
        case 2: return launch_force_k<2, MODE, EPS_I, DIRECT>(args, plan, stream);
        case 4: return launch_force_k<4, MODE, EPS_I, DIRECT>(args, plan, stream);
        default: return launch_force_k<8, MODE, EPS_I, DIRECT>(args, plan, stream);
    }
}

// counts stay 4096 below 2^31 so that tile-padded 32-bit particle indices cannot wrap inside the kernels
constexpr int64_t kMaxCount = (int64_t)INT32_MAX - 4096;
bool bad_count(int64_t n) { return n < 0 || n > kMaxCount; }

// Coincidence pre-pass (MODE_LIST): hash table over the j-positions, one sorted j-segment list per
// i-group of 32*K i-particles.  jp = packed j records, stride float4 each.  Three launches.
int coin_prepass(Workspace* ws, const nb::Plan& plan, int64_t n_i, const float* x_i, int64_t n_j, const float4* jp,
                 int stride, cudaStream_t stream, const int** lists_out, const int** flag_out) {
    const int group = 32 * plan.K;
    const int64_t n_groups = (int64_t)plan.tiles_i * plan.WI;        // every warp slot of the grid has a list
    uint32_t slots = 1024;
    while ((int64_t)slots < 2 * n_j) slots <<= 1;
    const size_t b_lists = ((size_t)(1 + n_groups * (1 + nb::kCoinCap)) * sizeof(int) + 255) / 256 * 256;
    int rc = ensure(&ws->coin, &ws->coin_bytes, b_lists + (size_t)slots * sizeof(uint32_t), stream);
    if (rc != NB_OK) return rc;
    int* flag = reinterpret_cast<int*>(ws->coin);
    int* lists = flag + 1;
    uint32_t* table = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(ws->coin) + b_lists);
    NB_CUDA(cudaMemsetAsync(ws->coin, 0, b_lists + (size_t)slots * sizeof(uint32_t), stream));
    nb::nb_coin_insert_kernel<<<(unsigned)((n_j + 255) / 256), 256, 0, stream>>>(jp, stride, (int)n_j, table, slots - 1, flag);
    NB_CUDA(cudaGetLastError());
    nb::nb_coin_probe_kernel<<<(unsigned)n_groups, group, 0, stream>>>(x_i, (int)n_i, jp, stride, table, slots - 1, lists);
    NB_CUDA(cudaGetLastError());
    t_launches += 2;
    *lists_out = lists;
    *flag_out = flag;
    return NB_OK;
}

// Which calls take the small-i-set kernel (nb_small.cuh): few i-particles, where nb_force_kernel's packing over i leaves
// a thread one dependent chain (thresholds from the scan in profiles/r02_small_calls.md).  NB_SMALL=0/1 forces.
bool use_small_path(const Knobs& kn, int64_t n_i, int64_t n_j) {
    if (kn.small >= 0) return kn.small != 0;
    if (kn.plan_set || kn.mask >= 0 || kn.fused >= 0 || kn.direct >= 0) return false;   // a switch of nb_force_kernel's paths is set
    return nb::small_by_default(n_i, n_j);
}

// pack (a1) when repack is true, then force (+ reduce).  The packed array lives in the workspace.
// eps2_i != nullptr: row f3, the softening of every i-particle comes from that device array and eps2 is ignored.
int force_impl(int64_t n_i, const float* x_i, int64_t n_j, const float* x_j, const float* m_j, float eps2,
               float* acc_out, float* pot_out, cudaStream_t stream, const float* eps2_i = nullptr,
               const float4* packed_j = nullptr) {
    // packed_j != nullptr: the caller already holds the 16-byte (x, y, z, m) records (nb_force_packed); x_j, m_j unused
    if (bad_count(n_i) || bad_count(n_j)) return NB_ERR_INVALID_VALUE;
    if (!eps2_i && (!(eps2 >= 0.0f) || !std::isfinite(eps2))) return NB_ERR_INVALID_VALUE;
    if (n_i > 0 && (!x_i || !acc_out)) return NB_ERR_INVALID_VALUE;
    if (n_j > 0 && !packed_j && (!x_j || !m_j)) return NB_ERR_INVALID_VALUE;
    if (packed_j && (reinterpret_cast<uintptr_t>(packed_j) & 15u)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_i == 0) return NB_OK;
    if (n_j == 0) {
        NB_CUDA(cudaMemsetAsync(acc_out, 0, sizeof(float) * 3 * (size_t)n_i, stream));
        if (pot_out) NB_CUDA(cudaMemsetAsync(pot_out, 0, sizeof(float) * (size_t)n_i, stream));
        return NB_OK;
    }
    const Knobs& kn = knobs();
    // Without phi no pair needs a mask when eps2 >= 2^-40: an unmasked coincident pair adds m u^3 * (+-0) = +-0 to a
    // (only phi would get m / eps), so a_i is bit for bit the masked loop's.  The list-mode kernel then runs with an
    // empty list: no pre-pass, the untested loop everywhere (nb_leapfrog_kdk: every evaluation but the last).
    const bool a_only = !pot_out && !eps2_i && eps2 >= kUnmaskedMinEps2 && kn.mask < 0;

    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;

    // Small i-sets: the kernel packed over j (nb_small.cuh), one launch, cluster + ticket reduction of the j-split.
    if (!eps2_i && use_small_path(kn, n_i, n_j)) {
        nb::SmallPlan sp = cached_small_plan(n_i, n_j, info.sm_count);
        if (kn.small_plan_set) {
            sp.NW = kn.sNW; sp.KI = kn.sKI; sp.LJ = kn.sLJ; sp.WJ = kn.sWJ; sp.S = kn.sS; sp.CS = kn.sCS;
            sp.tile_i = (sp.NW / sp.WJ) * sp.KI * (32 / sp.LJ);
            sp.tiles_i = (int)((n_i + sp.tile_i - 1) / sp.tile_i);
        }
        if (kn.small_pdl == 0) sp.pdl = 0;
        const int n_groups = sp.S / sp.CS;
        if (n_groups > 1) {
            rc = ensure(&ws->partial, &ws->partial_bytes, (size_t)n_groups * (size_t)n_i * sizeof(double4), stream);
            if (rc != NB_OK) return rc;
            const size_t need = (size_t)sp.tiles_i * sp.CS * sizeof(int);
            if (need > ws->tickets_bytes) {
                rc = ensure(&ws->tickets, &ws->tickets_bytes, need, stream);
                if (rc != NB_OK) return rc;
                NB_CUDA(cudaMemsetAsync(ws->tickets, 0, ws->tickets_bytes, stream));   // once per growth; kernels leave zeros
            }
        }
        nb::SmallArgs sa;
        sa.x_i = x_i;
        sa.xj_raw = packed_j ? nullptr : x_j;
        sa.mj_raw = packed_j ? nullptr : m_j;
        sa.jp = packed_j;
        sa.acc = acc_out;
        sa.pot = pot_out;
        sa.partial = reinterpret_cast<double4*>(ws->partial);
        sa.tickets = reinterpret_cast<int*>(ws->tickets);
        sa.n_i = (int)n_i;
        sa.n_j = (int)n_j;
        sa.S = sp.S;
        sa.eps2 = eps2;
        sa.flag_offset = 0;
        // coincident pairs: no mask at all without phi (eps2 >= 2^-40); else only the pairs marked while staged are masked
        // -- or every pair: eps2 < 2^-40 (an unmasked coincident pair would overflow), NB_SMALL_MASK=exact
        // (marking pays when a thread's loop is long: filter + tests cost ~1 us, the unmasked loop runs 10-15 % faster;
        //  measured on C2 24.65 -> 23.64 us per call, on C0 -- 64 pairs per thread -- nothing: profiles/r02_small_calls.md)
        const bool flag_pays = nb::small_flag_pays(sp, n_j);
        const int small_mode = a_only ? nb::SMALL_NONE
                               : (eps2 >= kUnmaskedMinEps2 && kn.small_mask != nb::SMALL_EXACT && (flag_pays || kn.small_mask == nb::SMALL_FLAG))
                                     ? nb::SMALL_FLAG : nb::SMALL_EXACT;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (t_profile) {
            NB_CUDA(cudaEventCreate(&e0));
            NB_CUDA(cudaEventCreate(&e1));
            NB_CUDA(cudaEventRecord(e0, stream));
        }
        NB_CUDA(nb::small_launch(sp, sa, small_mode, stream));
        if (t_profile) {
            NB_CUDA(cudaEventRecord(e1, stream));
            t_events.emplace_back(e0, e1);
        }
        ++t_launches;
        return NB_OK;
    }

    const nb::Plan plan = cached_plan(n_i, n_j, info.sm_count);
    const int mode = pick_mode(n_i, n_j, eps2_i ? 1.0f : eps2, eps2_i == nullptr);
    // Small calls whose per-warp-group j sub-range fits its shared-memory ring whole: the force kernel packs the
    // sub-range itself, one launch fewer.  NB_DIRECT=0 (nb_debug.h) disables it (tests compare).
    const int64_t sub_max = (n_j + (int64_t)plan.S * plan.WJ - 1) / ((int64_t)plan.S * plan.WJ);
    const bool direct = !packed_j && !eps2_i && mode != nb::MODE_LIST && sub_max <= (int64_t)plan.tile_j * plan.stages &&
                        kn.direct != 0;
    if (!packed_j && !direct) {                                        // the packed records live in the workspace
        rc = ensure(&ws->jp, &ws->jp_bytes, (size_t)n_j * sizeof(float4), stream);
        if (rc != NB_OK) return rc;
    }
    // second pass: fused into the force kernel or a separate launch (nb_plan.h: fused_second_pass); NB_FUSED_REDUCE forces
    const bool fused_reduce = kn.fused >= 0 ? (kn.fused != 0) : nb::fused_second_pass(plan.tile_i, plan.S);
    if (plan.S > 1) {
        rc = ensure(&ws->partial, &ws->partial_bytes, (size_t)plan.S * (size_t)n_i * sizeof(double4), stream);
        if (rc != NB_OK) return rc;
        if (fused_reduce && (size_t)plan.tiles_i * sizeof(int) > ws->tickets_bytes) {
            rc = ensure(&ws->tickets, &ws->tickets_bytes, (size_t)plan.tiles_i * sizeof(int), stream);
            if (rc != NB_OK) return rc;
            NB_CUDA(cudaMemsetAsync(ws->tickets, 0, ws->tickets_bytes, stream));   // once per growth; kernels leave zeros
        }
    }
    const float4* jp = packed_j ? packed_j : reinterpret_cast<const float4*>(ws->jp);
    if (!packed_j && !direct) {   // a1: j-pack
        const int threads = 256;
        const int blocks = (int)((n_j + threads - 1) / threads);
        nb::nb_pack_j_kernel<<<blocks, threads, 0, stream>>>(x_j, m_j, (int)n_j, reinterpret_cast<float4*>(ws->jp));
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }

    nb::ForceArgs args;
    args.x_i = x_i;
    args.eps2_i = eps2_i;
    args.jp = jp;
    args.xj_raw = direct ? x_j : nullptr;
    args.mj_raw = direct ? m_j : nullptr;
    args.acc = acc_out;
    args.pot = pot_out;
    args.partial = reinterpret_cast<double4*>(ws->partial);
    args.tickets = (plan.S > 1 && fused_reduce) ? reinterpret_cast<int*>(ws->tickets) : nullptr;
    args.n_i = (int)n_i;
    args.n_j = (int)n_j;
    args.S = plan.S;
    args.eps2 = eps2;
    args.coin_lists = nullptr;
    args.coin_flag = nullptr;
    args.i_off = args.j_off = args.tile_start = args.cta_batch = args.j_index = nullptr;
    args.n_batch = 0;
    if (direct) {                                                      // small call: one launch (packs its own j)
        rc = (mode == nb::MODE_BLOOM) ? launch_force<nb::MODE_BLOOM, false, true>(args, plan, stream)
                                      : launch_force<nb::MODE_EXACT, false, true>(args, plan, stream);
    } else if (a_only) {
        rc = (plan.K == 8) ? launch_force_nophi(args, plan, stream) : launch_force<nb::MODE_LIST>(args, plan, stream);
    } else if (mode == nb::MODE_LIST) {
        rc = coin_prepass(ws, plan, n_i, x_i, n_j, jp, 1, stream, &args.coin_lists, &args.coin_flag);
        if (rc != NB_OK) return rc;
        if (eps2_i) rc = launch_force<nb::MODE_LIST, true>(args, plan, stream);
        else if (!pot_out && plan.K == 8) rc = launch_force_nophi(args, plan, stream);
        else rc = launch_force<nb::MODE_LIST>(args, plan, stream);
    } else if (eps2_i) {
        rc = launch_force<nb::MODE_EXACT, true>(args, plan, stream);
    } else if (mode == nb::MODE_BLOOM) {
        rc = launch_force<nb::MODE_BLOOM>(args, plan, stream);
    } else {
        rc = launch_force<nb::MODE_EXACT>(args, plan, stream);
    }
    if (rc != NB_OK) return rc;

    if (plan.S > 1 && !fused_reduce) {
        const int threads = 128;
        const int blocks = (int)((n_i + threads - 1) / threads);
        nb::nb_reduce_kernel<<<blocks, threads, 0, stream>>>(reinterpret_cast<const double4*>(ws->partial), (int)n_i,
                                                             plan.S, acc_out, pot_out);
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    return NB_OK;
}


// ------------------------------------------------------------------ row f1: force + jerk + potential
nb::Plan hermite_plan(int64_t n_i, int64_t n_j, int sm_count) {
    return nb::make_plan(n_i, n_j, sm_count, 4, kHermiteInstPerPair, kHermitePartialBytes);
}

template <int K, int WI, int WJ, int STAGES, int MODE, bool PHI = true>
int launch_hermite_inst(const nb::HermiteArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    constexpr int TJ = 256;
    constexpr size_t ring = (size_t)WJ * STAGES * TJ * 32;
    constexpr size_t red = (WJ > 1) ? (size_t)WJ * K * nb::kHermiteAcc * (WI * 32) * sizeof(double) : 0;
    constexpr size_t bloom = (MODE == nb::MODE_BLOOM) ? (size_t)WI * nb::kBloomWords * sizeof(uint32_t) : 0;
    constexpr size_t smem = (ring + bloom > red ? ring + bloom : red) + 2 * WJ * STAGES * sizeof(uint64_t) + 128;
    static std::atomic<uint64_t> configured{0};
    return launch_dominant(nb::nb_hermite_kernel<K, WI, WJ, TJ, STAGES, MODE, PHI>, &configured,
                           dim3((unsigned)plan.tiles_i, (unsigned)plan.S, 1), 32 * WI * WJ, smem, stream, args);
}

template <int K, int MODE>
int launch_hermite_k(const nb::HermiteArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    switch (plan.WJ) {
        case 1: return launch_hermite_inst<K, 8, 1, 4, MODE>(args, plan, stream);
        case 2: return launch_hermite_inst<K, 4, 2, 4, MODE>(args, plan, stream);
        case 4: return launch_hermite_inst<K, 2, 4, 3, MODE>(args, plan, stream);
        default: return launch_hermite_inst<K, 1, 8, 3, MODE>(args, plan, stream);
    }
}

// pot_out == NULL (nb_hermite4: every evaluation but the last): 26 instructions per pair, K = 4, list and Bloom modes
template <int MODE>
int launch_hermite_nophi(const nb::HermiteArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    switch (plan.WJ) {
        case 1: return launch_hermite_inst<4, 8, 1, 4, MODE, false>(args, plan, stream);
        case 2: return launch_hermite_inst<4, 4, 2, 4, MODE, false>(args, plan, stream);
        case 4: return launch_hermite_inst<4, 2, 4, 3, MODE, false>(args, plan, stream);
        default: return launch_hermite_inst<4, 1, 8, 3, MODE, false>(args, plan, stream);
    }
}

template <int MODE>
int launch_hermite(const nb::HermiteArgs& args, const nb::Plan& plan, cudaStream_t stream) {
    return plan.K == 2 ? launch_hermite_k<2, MODE>(args, plan, stream) : launch_hermite_k<4, MODE>(args, plan, stream);
}

int force_jerk_impl(int64_t n_i, const float* x_i, const float* v_i, int64_t n_j, const float* x_j, const float* v_j,
                    const float* m_j, float eps2, float* acc_out, float* jerk_out, float* pot_out, cudaStream_t stream,
                    bool prepacked = false) {   // prepacked: the caller has filled the workspace's packed j records
    if (bad_count(n_i) || bad_count(n_j)) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2)) return NB_ERR_INVALID_VALUE;
    if (n_i > 0 && (!x_i || !v_i || !acc_out || !jerk_out)) return NB_ERR_INVALID_VALUE;
    if (n_j > 0 && (!x_j || !v_j || !m_j)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_i == 0) return NB_OK;
    if (n_j == 0) {
        NB_CUDA(cudaMemsetAsync(acc_out, 0, sizeof(float) * 3 * (size_t)n_i, stream));
        NB_CUDA(cudaMemsetAsync(jerk_out, 0, sizeof(float) * 3 * (size_t)n_i, stream));
        if (pot_out) NB_CUDA(cudaMemsetAsync(pot_out, 0, sizeof(float) * (size_t)n_i, stream));
        return NB_OK;
    }
    const Knobs& kn = knobs();
    const nb::Plan plan = cached_plan(n_i, n_j, info.sm_count, true);
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    // Small i-sets: the kernel packed over j (nb_small_hermite.cuh), one launch (it packs the j-records itself unless the
    // caller -- a Hermite step's predictor -- already has)
    if (kn.small_jerk >= 0 ? (kn.small_jerk != 0)
                           : (!kn.plan_set && kn.mask < 0 && kn.fused < 0 && nb::small_jerk_by_default(n_i, n_j, prepacked))) {
        nb::SmallPlan sp = cached_small_jerk_plan(n_i, n_j, info.sm_count);
        if (kn.small_jerk_plan_set) {
            sp.NW = kn.jNW; sp.KI = 1; sp.LJ = kn.jLJ; sp.WJ = kn.jWJ; sp.S = kn.jS; sp.CS = kn.jCS;
            sp.tile_i = (sp.NW / sp.WJ) * (32 / sp.LJ);
            sp.tiles_i = (int)((n_i + sp.tile_i - 1) / sp.tile_i);
        }
        if (kn.small_pdl == 0) sp.pdl = 0;
        const int n_groups = sp.S / sp.CS;
        if (n_groups > 1) {
            rc = ensure(&ws->hpartial, &ws->hpartial_bytes, (size_t)n_groups * (size_t)n_i * nb::kHermiteAcc * sizeof(double), stream);
            if (rc != NB_OK) return rc;
            const size_t need = (size_t)sp.tiles_i * sp.CS * sizeof(int);
            if (need > ws->tickets_bytes) {
                rc = ensure(&ws->tickets, &ws->tickets_bytes, need, stream);
                if (rc != NB_OK) return rc;
                NB_CUDA(cudaMemsetAsync(ws->tickets, 0, ws->tickets_bytes, stream));   // once per growth; kernels leave zeros
            }
        }
        nb::SmallHermiteArgs sa;
        sa.x_i = x_i;
        sa.v_i = v_i;
        sa.jp = prepacked ? reinterpret_cast<const float4*>(ws->jp2) : nullptr;   // not packed yet: the kernel reads the three arrays
        sa.xj_raw = x_j;
        sa.vj_raw = v_j;
        sa.mj_raw = m_j;
        sa.acc = acc_out;
        sa.jerk = jerk_out;
        sa.pot = pot_out;
        sa.partial = reinterpret_cast<double*>(ws->hpartial);
        sa.tickets = reinterpret_cast<int*>(ws->tickets);
        sa.n_i = (int)n_i;
        sa.n_j = (int)n_j;
        sa.S = sp.S;
        sa.eps2 = eps2;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (t_profile) {
            NB_CUDA(cudaEventCreate(&e0));
            NB_CUDA(cudaEventCreate(&e1));
            NB_CUDA(cudaEventRecord(e0, stream));
        }
        NB_CUDA(nb::small_hermite_launch(sp, sa, stream));
        if (t_profile) {
            NB_CUDA(cudaEventRecord(e1, stream));
            t_events.emplace_back(e0, e1);
        }
        ++t_launches;
        return NB_OK;
    }
    rc = ensure(&ws->jp2, &ws->jp2_bytes, (size_t)n_j * 2 * sizeof(float4), stream);
    if (rc != NB_OK) return rc;
    // second pass: fused into the kernel (small tiles) or a separate launch, as for nb_force; NB_FUSED_REDUCE=0/1 forces
    const int mode = pick_mode(n_i, n_j, eps2, true, kListMinPairsJerk);
    const bool fused_reduce = plan.S > 1 && mode == nb::MODE_EXACT &&      // only the masked (small-call) kernels carry the ticket code
                              (kn.fused >= 0 ? (kn.fused != 0) : nb::fused_second_pass(plan.tile_i, plan.S, kHermitePartialBytes));
    if (plan.S > 1) {
        rc = ensure(&ws->hpartial, &ws->hpartial_bytes, (size_t)plan.S * (size_t)n_i * nb::kHermiteAcc * sizeof(double), stream);
        if (rc != NB_OK) return rc;
        if (fused_reduce && (size_t)plan.tiles_i * sizeof(int) > ws->tickets_bytes) {
            rc = ensure(&ws->tickets, &ws->tickets_bytes, (size_t)plan.tiles_i * sizeof(int), stream);
            if (rc != NB_OK) return rc;
            NB_CUDA(cudaMemsetAsync(ws->tickets, 0, ws->tickets_bytes, stream));   // once per growth; kernels leave zeros
        }
    }
    if (!prepacked) {
        nb::nb_pack_jv_kernel<<<(unsigned)((n_j + 255) / 256), 256, 0, stream>>>(x_j, v_j, m_j, (int)n_j,
                                                                                  reinterpret_cast<float4*>(ws->jp2));
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }

    nb::HermiteArgs args;
    args.x_i = x_i;
    args.v_i = v_i;
    args.jp = reinterpret_cast<const float4*>(ws->jp2);
    args.acc = acc_out;
    args.jerk = jerk_out;
    args.pot = pot_out;
    args.partial = reinterpret_cast<double*>(ws->hpartial);
    args.tickets = fused_reduce ? reinterpret_cast<int*>(ws->tickets) : nullptr;
    args.coin_lists = nullptr;
    args.coin_flag = nullptr;
    args.n_i = (int)n_i;
    args.n_j = (int)n_j;
    args.S = plan.S;
    args.eps2 = eps2;
    // small calls mask every pair, mid-size ones test every block against a Bloom filter, large ones use the coincidence lists
    if (mode == nb::MODE_LIST) {
        rc = coin_prepass(ws, plan, n_i, x_i, n_j, args.jp, 2, stream, &args.coin_lists, &args.coin_flag);
        if (rc != NB_OK) return rc;
        rc = (!pot_out && plan.K == 4) ? launch_hermite_nophi<nb::MODE_LIST>(args, plan, stream) : launch_hermite<nb::MODE_LIST>(args, plan, stream);
    } else if (mode == nb::MODE_BLOOM) {
        rc = (!pot_out && plan.K == 4) ? launch_hermite_nophi<nb::MODE_BLOOM>(args, plan, stream) : launch_hermite<nb::MODE_BLOOM>(args, plan, stream);
    } else {
        rc = launch_hermite<nb::MODE_EXACT>(args, plan, stream);
    }
    if (rc != NB_OK) return rc;
    if (plan.S > 1 && !fused_reduce) {
        nb::nb_hermite_reduce_kernel<<<(unsigned)((n_i + 127) / 128), 128, 0, stream>>>(
            reinterpret_cast<const double*>(ws->hpartial), (int)n_i, plan.S, acc_out, jerk_out, pot_out);
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    return NB_OK;
}


// ------------------------------------------------------------------ row f2: many small sub-problems in one launch
// i-tile of a batched call: 64 G particles per CTA.  Measured on tree lists (groups of 32..256, lists of 2000..6000):
// small tiles win -- less padding in every group's last tile, and several CTAs per SM overlap their prologues.
int batched_groups(int64_t n_i_total, int64_t n_batch) {
    const double mean = (double)n_i_total / (double)(n_batch > 0 ? n_batch : 1);
    if (const int t = knobs().batch_tile) return t / 64;            // NB_BATCH_TILE (nb_debug.h)
    if (mean <= 384.0) return 1;
    if (mean <= 1024.0) return 2;
    return 4;
}

template <bool MASKED, int G, int STAGES, bool INDEXED>
int launch_batched_inst(const nb::ForceArgs& args, unsigned max_ctas, cudaStream_t stream) {
    constexpr size_t ring = (size_t)8 * STAGES * 256 * 16;
    constexpr size_t red = (size_t)8 * (2 * G) * 4 * 32 * sizeof(double);
    constexpr size_t smem = (ring > red ? ring : red) + 8 * STAGES * sizeof(uint64_t) + 128;
    static std::atomic<uint64_t> configured{0};
    return launch_dominant(nb::nb_batched_kernel<MASKED, G, STAGES, INDEXED>, &configured, dim3(max_ctas, 1, 1), 256, smem, stream, args);
}

template <bool MASKED, bool INDEXED>
int launch_batched(const nb::ForceArgs& args, int groups, unsigned max_ctas, cudaStream_t stream) {
    switch (groups) {
        case 1: return launch_batched_inst<MASKED, 1, 2, INDEXED>(args, max_ctas, stream);  // 64 KB of rings, 2 CTAs per SM
        case 2: return launch_batched_inst<MASKED, 2, 3, INDEXED>(args, max_ctas, stream);
        default: return launch_batched_inst<MASKED, 4, 3, INDEXED>(args, max_ctas, stream);
    }
}

}  // namespace

extern "C" {

}  // extern "C"

namespace {
// packed_j != nullptr: the caller holds the list records as 16-byte (x, y, z, m) rows already (nb_force_batched_packed)
// j_index != nullptr: the lists are indices into the packed particle array packed_j [n_p] (nb_force_batched_indexed);
// n_j_total is then the number of list entries
int force_batched_impl(int64_t n_batch, const int32_t* i_offsets, const int32_t* j_offsets, int64_t n_i_total,
                       const float* x_i, int64_t n_j_total, const float* x_j, const float* m_j, const float4* packed_j,
                       float eps2, float* acc_out, float* pot_out, void* stream_, const int32_t* j_index = nullptr) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n_batch) || bad_count(n_i_total) || bad_count(n_j_total)) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2)) return NB_ERR_INVALID_VALUE;
    if (n_batch > 0 && (!i_offsets || !j_offsets)) return NB_ERR_INVALID_VALUE;
    if (n_i_total > 0 && (!x_i || !acc_out)) return NB_ERR_INVALID_VALUE;
    if (n_j_total > 0 && !packed_j && (!x_j || !m_j)) return NB_ERR_INVALID_VALUE;
    if (packed_j && (reinterpret_cast<uintptr_t>(packed_j) & 15u)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_batch == 0 || n_i_total == 0) return NB_OK;
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    if (!packed_j) {
        rc = ensure(&ws->jp, &ws->jp_bytes, (size_t)(n_j_total > 0 ? n_j_total : 1) * sizeof(float4), stream);
        if (rc != NB_OK) return rc;
    }
    const int groups = batched_groups(n_i_total, n_batch);
    const int tile = 64 * groups;
    // sum_b ceil(n_i(b) / tile) <= n_i_total / tile + n_batch
    const int64_t max_ctas = n_i_total / tile + n_batch;
    if (max_ctas > (int64_t)INT32_MAX) return NB_ERR_INVALID_VALUE;
    rc = ensure(&ws->tiles, &ws->tiles_bytes, (size_t)(n_batch + 1 + max_ctas) * sizeof(int), stream);
    if (rc != NB_OK) return rc;
    if (n_j_total > 0 && !packed_j) {
        nb::nb_pack_j_kernel<<<(unsigned)((n_j_total + 255) / 256), 256, 0, stream>>>(x_j, m_j, (int)n_j_total,
                                                                                      reinterpret_cast<float4*>(ws->jp));
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    int* tile_start = reinterpret_cast<int*>(ws->tiles);
    int* cta_batch = tile_start + n_batch + 1;
    nb::nb_batch_scan_kernel<<<1, 1024, 0, stream>>>(i_offsets, (int)n_batch, tile, tile_start, cta_batch);
    NB_CUDA(cudaGetLastError());
    ++t_launches;

    nb::ForceArgs args;
    args.x_i = x_i;
    args.eps2_i = nullptr;
    args.jp = packed_j ? packed_j : reinterpret_cast<const float4*>(ws->jp);
    args.xj_raw = args.mj_raw = nullptr;
    args.acc = acc_out;
    args.pot = pot_out;
    args.partial = nullptr;
    args.tickets = nullptr;
    args.coin_lists = nullptr;
    args.coin_flag = nullptr;
    args.j_index = j_index;
    args.i_off = i_offsets;
    args.j_off = j_offsets;
    args.tile_start = tile_start;
    args.cta_batch = cta_batch;
    args.n_batch = (int)n_batch;
    args.n_i = (int)n_i_total;
    args.n_j = (int)n_j_total;
    args.S = 1;
    args.eps2 = eps2;
    // every pair masked -- unless phi is not wanted and eps2 >= 2^-40, where no pair needs the mask (see force_impl)
    const bool a_only = !pot_out && eps2 >= kUnmaskedMinEps2 && knobs().mask < 0;
    if (j_index)
        return a_only ? launch_batched<false, true>(args, groups, (unsigned)max_ctas, stream)
                      : launch_batched<true, true>(args, groups, (unsigned)max_ctas, stream);
    return a_only ? launch_batched<false, false>(args, groups, (unsigned)max_ctas, stream)
                  : launch_batched<true, false>(args, groups, (unsigned)max_ctas, stream);
}
}  // namespace

extern "C" {

int nb_force_batched(int64_t n_batch, const int32_t* i_offsets, const int32_t* j_offsets, int64_t n_i_total,
                     const float* x_i, int64_t n_j_total, const float* x_j, const float* m_j, float eps2,
                     float* acc_out, float* pot_out, void* stream) {
    return force_batched_impl(n_batch, i_offsets, j_offsets, n_i_total, x_i, n_j_total, x_j, m_j, nullptr, eps2, acc_out, pot_out, stream);
}

int nb_force_batched_indexed(int64_t n_batch, const int32_t* i_offsets, const int32_t* j_offsets, int64_t n_i_total,
                             const float* x_i, int64_t n_list_total, const int32_t* j_index, int64_t n_p, const float* xm_p,
                             float eps2, float* acc_out, float* pot_out, void* stream) {
    if (bad_count(n_p) || (n_list_total > 0 && (!j_index || !xm_p || n_p < 1))) return NB_ERR_INVALID_VALUE;
    static const float4 dummy = {0.f, 0.f, 0.f, 0.f};
    static const int32_t dummy_index = 0;
    return force_batched_impl(n_batch, i_offsets, j_offsets, n_i_total, x_i, n_list_total, nullptr, nullptr,
                              xm_p ? reinterpret_cast<const float4*>(xm_p) : &dummy, eps2, acc_out, pot_out, stream,
                              j_index ? j_index : &dummy_index);
}

int nb_force_batched_packed(int64_t n_batch, const int32_t* i_offsets, const int32_t* j_offsets, int64_t n_i_total,
                            const float* x_i, int64_t n_j_total, const float* xm_j, float eps2,
                            float* acc_out, float* pot_out, void* stream) {
    if (n_j_total > 0 && !xm_j) return NB_ERR_INVALID_VALUE;
    static const float4 dummy = {0.f, 0.f, 0.f, 0.f};
    return force_batched_impl(n_batch, i_offsets, j_offsets, n_i_total, x_i, n_j_total, nullptr, nullptr,
                              xm_j ? reinterpret_cast<const float4*>(xm_j) : &dummy, eps2, acc_out, pot_out, stream);
}

int nb_force_jerk(int64_t n_i, const float* x_i, const float* v_i, int64_t n_j, const float* x_j, const float* v_j,
                  const float* m_j, float eps2, float* acc_out, float* jerk_out, float* pot_out, void* stream) {
    t_launches = 0;
    return force_jerk_impl(n_i, x_i, v_i, n_j, x_j, v_j, m_j, eps2, acc_out, jerk_out, pot_out,
                           reinterpret_cast<cudaStream_t>(stream));
}

int nb_force_jerk_host(int64_t n_i, const float* x_i, const float* v_i, int64_t n_j, const float* x_j, const float* v_j,
                       const float* m_j, float eps2, float* acc_out, float* jerk_out, float* pot_out) {
    t_launches = 0;
    if (bad_count(n_i) || bad_count(n_j)) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2)) return NB_ERR_INVALID_VALUE;
    if (n_i > 0 && (!x_i || !v_i || !acc_out || !jerk_out)) return NB_ERR_INVALID_VALUE;
    if (n_j > 0 && (!x_j || !v_j || !m_j)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_i == 0) return NB_OK;
    cudaStream_t stream = nullptr;   // legacy default stream
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    auto up = [](size_t b) { return (b + 255) / 256 * 256; };
    const bool aliased = (x_i == x_j && v_i == v_j && n_i <= n_j);
    const size_t b_j3 = up(sizeof(float) * 3 * (size_t)n_j), b_mj = up(sizeof(float) * (size_t)n_j);
    const size_t b_i3 = up(sizeof(float) * 3 * (size_t)n_i), b_pot = up(sizeof(float) * (size_t)n_i);
    const size_t total = 2 * b_j3 + b_mj + (aliased ? 0 : 2 * b_i3) + 2 * b_i3 + b_pot + 256;
    rc = ensure(&ws->stage, &ws->stage_bytes, total, stream);
    if (rc != NB_OK) return rc;
    char* p = reinterpret_cast<char*>(ws->stage);
    float* d_xj = reinterpret_cast<float*>(p); p += b_j3;
    float* d_vj = reinterpret_cast<float*>(p); p += b_j3;
    float* d_mj = reinterpret_cast<float*>(p); p += b_mj;
    float* d_xi = d_xj; float* d_vi = d_vj;
    if (!aliased) { d_xi = reinterpret_cast<float*>(p); p += b_i3; d_vi = reinterpret_cast<float*>(p); p += b_i3; }
    float* d_acc = reinterpret_cast<float*>(p); p += b_i3;
    float* d_jerk = reinterpret_cast<float*>(p); p += b_i3;
    float* d_pot = reinterpret_cast<float*>(p);
    if (n_j > 0) {                                                             // step (a): host -> device
        NB_CUDA(cudaMemcpyAsync(d_xj, x_j, sizeof(float) * 3 * (size_t)n_j, cudaMemcpyHostToDevice, stream));
        NB_CUDA(cudaMemcpyAsync(d_vj, v_j, sizeof(float) * 3 * (size_t)n_j, cudaMemcpyHostToDevice, stream));
        NB_CUDA(cudaMemcpyAsync(d_mj, m_j, sizeof(float) * (size_t)n_j, cudaMemcpyHostToDevice, stream));
    }
    if (!aliased) {
        NB_CUDA(cudaMemcpyAsync(d_xi, x_i, sizeof(float) * 3 * (size_t)n_i, cudaMemcpyHostToDevice, stream));
        NB_CUDA(cudaMemcpyAsync(d_vi, v_i, sizeof(float) * 3 * (size_t)n_i, cudaMemcpyHostToDevice, stream));
    }
    rc = force_jerk_impl(n_i, d_xi, d_vi, n_j, d_xj, d_vj, d_mj, eps2, d_acc, d_jerk, pot_out ? d_pot : nullptr, stream);
    if (rc != NB_OK) return rc;
    NB_CUDA(cudaMemcpyAsync(acc_out, d_acc, sizeof(float) * 3 * (size_t)n_i, cudaMemcpyDeviceToHost, stream));   // step (l)
    NB_CUDA(cudaMemcpyAsync(jerk_out, d_jerk, sizeof(float) * 3 * (size_t)n_i, cudaMemcpyDeviceToHost, stream));
    if (pot_out) NB_CUDA(cudaMemcpyAsync(pot_out, d_pot, sizeof(float) * (size_t)n_i, cudaMemcpyDeviceToHost, stream));
    NB_CUDA(cudaStreamSynchronize(stream));
    return NB_OK;
}

int nb_plan_query_jerk(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]) {
    if (!out || bad_count(n_i) || bad_count(n_j) || n_i < 1 || n_j < 1) return NB_ERR_INVALID_VALUE;
    const nb::Plan p = hermite_plan(n_i, n_j, sm_count);
    out[0] = p.K; out[1] = p.WI; out[2] = p.WJ; out[3] = p.S;
    out[4] = p.tiles_i; out[5] = p.tile_i; out[6] = 256; out[7] = (p.WJ <= 2) ? 4 : 3;
    return NB_OK;
}

int nb_force(int64_t n_i, const float* x_i, int64_t n_j, const float* x_j, const float* m_j, float eps2,
             float* acc_out, float* pot_out, void* stream) {
    t_launches = 0;
    return force_impl(n_i, x_i, n_j, x_j, m_j, eps2, acc_out, pot_out, reinterpret_cast<cudaStream_t>(stream));
}

int nb_force_eps_i(int64_t n_i, const float* x_i, const float* eps2_i, int64_t n_j, const float* x_j, const float* m_j,
                   float* acc_out, float* pot_out, void* stream) {
    t_launches = 0;
    if (n_i > 0 && !eps2_i) return NB_ERR_INVALID_VALUE;
    static const float dummy = 0.0f;
    return force_impl(n_i, x_i, n_j, x_j, m_j, 0.0f, acc_out, pot_out, reinterpret_cast<cudaStream_t>(stream),
                      eps2_i ? eps2_i : &dummy);
}

}  // extern "C"

namespace {
// the cunbody_api call for a pipeline P on device rows
template <class P>
int cunbody_call(const float* p_xj, const float* p_xi, float* p_fi, int64_t ni, int64_t nj, cudaStream_t stream) {
    t_launches = 0;
    if (bad_count(ni) || bad_count(nj)) return NB_ERR_INVALID_VALUE;
    if (ni > 0 && (!p_xi || !p_fi)) return NB_ERR_INVALID_VALUE;
    if (nj > 0 && !p_xj) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (ni == 0) return NB_OK;
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    const size_t need = nj > 0 ? nb::pipeline_workspace_bytes<P>(ni, nj, info.sm_count) : 0;
    if (need) {
        rc = ensure(&ws->pipe, &ws->pipe_bytes, need, stream);
        if (rc != NB_OK) return rc;
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (t_profile) {                                                   // brackets the pair kernel and its second pass
        NB_CUDA(cudaEventCreate(&e0));
        NB_CUDA(cudaEventCreate(&e1));
        NB_CUDA(cudaEventRecord(e0, stream));
    }
    NB_CUDA(nb::pipeline_run<P>(p_xj, p_xi, p_fi, ni, nj, ws->pipe, info.sm_count, stream));
    if (t_profile) {
        NB_CUDA(cudaEventRecord(e1, stream));
        t_events.emplace_back(e0, e1);
    }
    t_launches = (nj > 0) ? (nb::pipeline_chunks<P>(ni, nj, info.sm_count) > 1 ? 2 : 1) : 0;
    return NB_OK;
}
}  // namespace

extern "C" {

int nb_cunbody_force(const float* p_xj, const float* p_xi, float* p_fi, int64_t ni, int64_t nj, void* stream) {
    return cunbody_call<nb::PipelineForceA3>(p_xj, p_xi, p_fi, ni, nj, reinterpret_cast<cudaStream_t>(stream));
}

int nb_cunbody_force_jerk_pot(const float* p_xj, const float* p_xi, float* p_fi, int64_t ni, int64_t nj, void* stream) {
    return cunbody_call<nb::PipelineForceJerkPotA4>(p_xj, p_xi, p_fi, ni, nj, reinterpret_cast<cudaStream_t>(stream));
}

int nb_cunbody_lennard_jones(const float* p_xj, const float* p_xi, float* p_fi, int64_t ni, int64_t nj, void* stream) {
    return cunbody_call<nb::PipelineLennardJones>(p_xj, p_xi, p_fi, ni, nj, reinterpret_cast<cudaStream_t>(stream));
}

int nb_pack_j(int64_t n_j, const float* x_j, const float* m_j, float* xm_out, void* stream) {
    t_launches = 0;
    if (bad_count(n_j)) return NB_ERR_INVALID_VALUE;
    if (n_j > 0 && (!x_j || !m_j || !xm_out)) return NB_ERR_INVALID_VALUE;
    if (reinterpret_cast<uintptr_t>(xm_out) & 15u) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_j == 0) return NB_OK;
    nb::nb_pack_j_kernel<<<(unsigned)((n_j + 255) / 256), 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(
        x_j, m_j, (int)n_j, reinterpret_cast<float4*>(xm_out));
    NB_CUDA(cudaGetLastError());
    ++t_launches;
    return NB_OK;
}

int nb_force_packed(int64_t n_i, const float* x_i, int64_t n_j, const float* xm_j, float eps2, float* acc_out,
                    float* pot_out, void* stream) {
    t_launches = 0;
    if (n_j > 0 && !xm_j) return NB_ERR_INVALID_VALUE;
    static const float4 dummy = {0.f, 0.f, 0.f, 0.f};
    return force_impl(n_i, x_i, n_j, nullptr, nullptr, eps2, acc_out, pot_out, reinterpret_cast<cudaStream_t>(stream),
                      nullptr, xm_j ? reinterpret_cast<const float4*>(xm_j) : &dummy);
}

int nb_force_host(int64_t n_i, const float* x_i, int64_t n_j, const float* x_j, const float* m_j, float eps2,
                  float* acc_out, float* pot_out) {
    t_launches = 0;
    if (bad_count(n_i) || bad_count(n_j)) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2)) return NB_ERR_INVALID_VALUE;
    if (n_i > 0 && (!x_i || !acc_out)) return NB_ERR_INVALID_VALUE;
    if (n_j > 0 && (!x_j || !m_j)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_i == 0) return NB_OK;
    cudaStream_t stream = nullptr;   // legacy default stream
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    auto up = [](size_t b) { return (b + 255) / 256 * 256; };
    const bool aliased = (x_i == x_j && n_i <= n_j);
    const size_t b_xj = up(sizeof(float) * 3 * (size_t)n_j), b_mj = up(sizeof(float) * (size_t)n_j);
    const size_t b_xi = aliased ? 0 : up(sizeof(float) * 3 * (size_t)n_i);
    const size_t b_acc = up(sizeof(float) * 3 * (size_t)n_i), b_pot = up(sizeof(float) * (size_t)n_i);
    rc = ensure(&ws->stage, &ws->stage_bytes, b_xj + b_mj + b_xi + b_acc + b_pot + 256, stream);
    if (rc != NB_OK) return rc;
    char* base = reinterpret_cast<char*>(ws->stage);
    float* d_xj = reinterpret_cast<float*>(base);
    float* d_mj = reinterpret_cast<float*>(base + b_xj);
    float* d_xi = aliased ? d_xj : reinterpret_cast<float*>(base + b_xj + b_mj);
    float* d_acc = reinterpret_cast<float*>(base + b_xj + b_mj + b_xi);
    float* d_pot = reinterpret_cast<float*>(base + b_xj + b_mj + b_xi + b_acc);
    // step (a): host -> device
    if (n_j > 0) {
        NB_CUDA(cudaMemcpyAsync(d_xj, x_j, sizeof(float) * 3 * (size_t)n_j, cudaMemcpyHostToDevice, stream));
        NB_CUDA(cudaMemcpyAsync(d_mj, m_j, sizeof(float) * (size_t)n_j, cudaMemcpyHostToDevice, stream));
    }
    if (!aliased) NB_CUDA(cudaMemcpyAsync(d_xi, x_i, sizeof(float) * 3 * (size_t)n_i, cudaMemcpyHostToDevice, stream));
    rc = force_impl(n_i, d_xi, n_j, d_xj, d_mj, eps2, d_acc, pot_out ? d_pot : nullptr, stream);
    if (rc != NB_OK) return rc;
    // step (l): device -> host
    NB_CUDA(cudaMemcpyAsync(acc_out, d_acc, sizeof(float) * 3 * (size_t)n_i, cudaMemcpyDeviceToHost, stream));
    if (pot_out) NB_CUDA(cudaMemcpyAsync(pot_out, d_pot, sizeof(float) * (size_t)n_i, cudaMemcpyDeviceToHost, stream));
    NB_CUDA(cudaStreamSynchronize(stream));
    return NB_OK;
}

int nb_leapfrog_kdk(int64_t n, float* x, float* v, const float* m, float eps2, float dt, int64_t n_steps,
                    float* acc_io, float* pot_out, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || n_steps < 0) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2) || !std::isfinite(dt)) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!x || !v || !m || !acc_io)) return NB_ERR_INVALID_VALUE;
    if (3 * n > (int64_t)INT32_MAX) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n == 0) return NB_OK;
    StreamDetour detour;                                               // a default stream: run on the device's private stream
    if (reinterpret_cast<uintptr_t>(stream) <= 2 && wants_step_graph(n, n_steps)) {
        rc = detour.begin(dev, stream, &stream);
        if (rc != NB_OK) return rc;
    }
    const int n3 = (int)(3 * n);
    const int threads = 256, blocks = (n3 + threads - 1) / threads;
    const float h = 0.5f * dt;
    // a0 = force(x0)
    // phi is only wanted at the final time: the evaluations before it run the 12-instruction loop without it
    rc = force_impl(n, x, n, x, m, eps2, acc_io, n_steps == 0 ? pot_out : nullptr, stream);
    if (rc != NB_OK) return rc;
    // Steps 1 .. n_steps-2 are identical launch sequences (fused kicks + drift, force without phi).  For small systems
    // a step is a few launches of ~10 us and the HOST becomes the limit (N = 2048: 13 us of enqueueing per step), so
    // those steps are captured once into a CUDA graph and replayed (N = 2048: 65 k -> see DESIGN.md steps/s).  Not
    // when the caller is itself capturing this stream, nor while kernel timing events are being recorded.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    NB_CUDA(cudaStreamIsCapturing(stream, &cap));
    const bool real_stream = reinterpret_cast<uintptr_t>(stream) > 2;   // the default streams cannot be captured
    const bool step_graph = real_stream && n_steps >= kStepGraphMinSteps && n <= 32768 && cap == cudaStreamCaptureStatusNone && !t_profile &&
                            knobs().step_graph != 0;                    // NB_STEP_GRAPH=0 (nb_debug.h): every step eagerly
    int64_t launches = t_launches;
    for (int64_t s = 0; s < n_steps; ++s) {
        // opening half-kick + drift; from the second step on it also carries the previous step's
        // closing half-kick (two separately rounded kicks, identical to the unfused sequence)
        if (step_graph && s == 2) {                                    // steps 0 and 1 ran eagerly: everything is warm
            cudaGraph_t graph = nullptr;
            cudaGraphExec_t exec = nullptr;
            // several steps per graph: one cudaGraphLaunch costs the host ~2 us, as much as a step of a small system
            const int64_t unroll = graph_steps(n_steps - 1 - s);
            NB_CUDA(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
            int64_t per_step = 0;
            for (int64_t u = 0; u < unroll && rc == NB_OK; ++u) {
                nb::nb_kick_drift_kernel<true><<<blocks, threads, 0, stream>>>(x, v, acc_io, n3, h, dt);
                t_launches = 0;
                rc = force_impl(n, x, n, x, m, eps2, acc_io, nullptr, stream);
                per_step = t_launches + 1;
            }
            cudaError_t ce = cudaStreamEndCapture(stream, &graph);
            if (rc != NB_OK || ce != cudaSuccess) {
                if (graph) (void)cudaGraphDestroy(graph);
                if (rc != NB_OK) return rc;
                t_last_cuda_error = (int)ce;
                return NB_ERR_CUDA;
            }
            NB_CUDA(cudaGraphInstantiate(&exec, graph, 0));
            const int64_t replays = (n_steps - 1 - s) / unroll;        // steps s .. n_steps-2, `unroll` at a time
            for (int64_t r = 0; r < replays; ++r) NB_CUDA(cudaGraphLaunch(exec, stream));
            (void)cudaGraphExecDestroy(exec);                          // freed by the runtime once the replays have run
            (void)cudaGraphDestroy(graph);
            launches += per_step * replays * unroll;
            s += replays * unroll;                                     // what is left (< unroll steps, and the last, which wants phi) runs eagerly
        }
        if (s == 0)
            nb::nb_kick_drift_kernel<false><<<blocks, threads, 0, stream>>>(x, v, acc_io, n3, h, dt);
        else
            nb::nb_kick_drift_kernel<true><<<blocks, threads, 0, stream>>>(x, v, acc_io, n3, h, dt);
        NB_CUDA(cudaGetLastError());
        t_launches = 0;
        rc = force_impl(n, x, n, x, m, eps2, acc_io, s + 1 == n_steps ? pot_out : nullptr, stream);
        if (rc != NB_OK) return rc;
        launches += t_launches + 1;
    }
    t_launches = launches;
    if (n_steps > 0) {
        nb::nb_kick_kernel<<<blocks, threads, 0, stream>>>(v, acc_io, n3, h);   // closing half-kick of the last step
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    return NB_OK;
}

int nb_kick_drift(int64_t n, float* x, float* v, const float* acc, float h, int n_kicks, float dt, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || 3 * n > (int64_t)INT32_MAX || (n_kicks != 1 && n_kicks != 2)) return NB_ERR_INVALID_VALUE;
    if (!std::isfinite(h) || !std::isfinite(dt)) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!x || !v || !acc)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n == 0) return NB_OK;
    const int n3 = (int)(3 * n), threads = 256, blocks = (n3 + threads - 1) / threads;
    if (n_kicks == 2) nb::nb_kick_drift_kernel<true><<<blocks, threads, 0, stream>>>(x, v, acc, n3, h, dt);
    else nb::nb_kick_drift_kernel<false><<<blocks, threads, 0, stream>>>(x, v, acc, n3, h, dt);
    NB_CUDA(cudaGetLastError());
    t_launches = 1;
    return NB_OK;
}

int nb_kick(int64_t n, float* v, const float* acc, float h, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || 3 * n > (int64_t)INT32_MAX || !std::isfinite(h)) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!v || !acc)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n == 0) return NB_OK;
    const int n3 = (int)(3 * n), threads = 256, blocks = (n3 + threads - 1) / threads;
    nb::nb_kick_kernel<<<blocks, threads, 0, stream>>>(v, acc, n3, h);
    NB_CUDA(cudaGetLastError());
    t_launches = 1;
    return NB_OK;
}

int nb_hermite4(int64_t n, float* x, float* v, const float* m, float eps2, float dt, int64_t n_steps, float* acc_io,
                float* jerk_io, float* pot_out, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || n_steps < 0) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2) || !std::isfinite(dt)) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!x || !v || !m || !acc_io || !jerk_io)) return NB_ERR_INVALID_VALUE;
    if (3 * n > (int64_t)INT32_MAX) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n == 0) return NB_OK;
    StreamDetour detour;                                               // a default stream: run on the device's private stream
    if (reinterpret_cast<uintptr_t>(stream) <= 2 && wants_step_graph(n, n_steps)) {
        rc = detour.begin(dev, stream, &stream);
        if (rc != NB_OK) return rc;
    }
    const int n3 = (int)(3 * n);
    const int threads = 256, blocks = (n3 + threads - 1) / threads;
    int64_t launches = 0;
    // a0, j0 = force_jerk(x0, v0)
    rc = force_jerk_impl(n, x, v, n, x, v, m, eps2, acc_io, jerk_io, n_steps == 0 ? pot_out : nullptr, stream);
    if (rc != NB_OK) return rc;
    launches += t_launches;
    if (n_steps == 0) return NB_OK;
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    const size_t b3 = ((size_t)n3 * sizeof(float) + 255) / 256 * 256;
    rc = ensure(&ws->hstate, &ws->hstate_bytes, 4 * b3, stream);
    if (rc != NB_OK) return rc;
    char* base = reinterpret_cast<char*>(ws->hstate);
    float* xp = reinterpret_cast<float*>(base);
    float* vp = reinterpret_cast<float*>(base + b3);
    float* a1 = reinterpret_cast<float*>(base + 2 * b3);
    float* j1 = reinterpret_cast<float*>(base + 3 * b3);
    // the prediction writes the packed j records of the predicted state itself (one launch fewer per step)
    rc = ensure(&ws->jp2, &ws->jp2_bytes, (size_t)n * 2 * sizeof(float4), stream);
    if (rc != NB_OK) return rc;
    float4* jp2 = reinterpret_cast<float4*>(ws->jp2);
    const int pblocks = (int)((n + threads - 1) / threads);
    // As in nb_leapfrog_kdk: on small systems the host's enqueueing is the limit, so the identical middle steps
    // (predict, force + jerk without phi, correct) are captured once into a CUDA graph and replayed.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    NB_CUDA(cudaStreamIsCapturing(stream, &cap));
    const bool real_stream = reinterpret_cast<uintptr_t>(stream) > 2;   // the default streams cannot be captured
    const bool step_graph = real_stream && n_steps >= kStepGraphMinSteps && n <= 32768 && cap == cudaStreamCaptureStatusNone && !t_profile &&
                            knobs().step_graph != 0;                    // NB_STEP_GRAPH=0 (nb_debug.h): every step eagerly
    // A step is two launches: force + jerk on the predicted state, then ONE kernel that corrects the step and predicts + packs
    // the next one (NB_HERMITE_FUSE=0, nb_debug.h: correct and predict as separate launches -- the same bits).
    const bool fuse = knobs().hermite_fuse != 0;
    nb::nb_hermite_predict_pack_kernel<<<pblocks, threads, 0, stream>>>(x, v, acc_io, jerk_io, m, xp, vp, jp2, (int)n, dt);
    NB_CUDA(cudaGetLastError());
    ++launches;
    auto launched = [&]() -> bool {                                    // NB_CUDA returns from the enclosing FUNCTION: not inside a lambda
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) t_last_cuda_error = (int)e;
        return e == cudaSuccess;
    };
    auto close_step = [&](bool last) -> int {                          // correct step s; unless it is the last, predict s + 1.  Launches, or -1
        if (!last && fuse) {
            nb::nb_hermite_correct_predict_pack_kernel<<<pblocks, threads, 0, stream>>>(x, v, acc_io, jerk_io, a1, j1, m, xp, vp, jp2, (int)n, dt);
            return launched() ? 1 : -1;
        }
        nb::nb_hermite_correct_kernel<<<blocks, threads, 0, stream>>>(x, v, acc_io, jerk_io, a1, j1, n3, dt);
        if (!launched()) return -1;
        if (last) return 1;
        nb::nb_hermite_predict_pack_kernel<<<pblocks, threads, 0, stream>>>(x, v, acc_io, jerk_io, m, xp, vp, jp2, (int)n, dt);
        return launched() ? 2 : -1;
    };
    for (int64_t s = 0; s < n_steps; ++s) {
        if (step_graph && s == 2 && n_steps - 1 - s > 0) {             // steps 0 and 1 ran eagerly: everything is warm
            cudaGraph_t graph = nullptr;
            cudaGraphExec_t exec = nullptr;
            const int64_t unroll = graph_steps(n_steps - 1 - s);       // several steps per graph, as nb_leapfrog_kdk
            NB_CUDA(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
            int64_t per_step = 0;
            for (int64_t u = 0; u < unroll && rc == NB_OK; ++u) {
                t_launches = 0;
                rc = force_jerk_impl(n, xp, vp, n, xp, vp, m, eps2, a1, j1, nullptr, stream, true);
                per_step = t_launches;
                if (rc == NB_OK) {
                    const int k = close_step(false);
                    if (k < 0) rc = NB_ERR_CUDA; else per_step += k;
                }
            }
            cudaError_t ce = cudaStreamEndCapture(stream, &graph);
            if (rc != NB_OK || ce != cudaSuccess) {
                if (graph) (void)cudaGraphDestroy(graph);
                if (rc != NB_OK) return rc;
                t_last_cuda_error = (int)ce;
                return NB_ERR_CUDA;
            }
            NB_CUDA(cudaGraphInstantiate(&exec, graph, 0));
            const int64_t replays = (n_steps - 1 - s) / unroll;        // steps s .. n_steps-2, `unroll` at a time
            for (int64_t r = 0; r < replays; ++r) NB_CUDA(cudaGraphLaunch(exec, stream));
            (void)cudaGraphExecDestroy(exec);                          // freed by the runtime once the replays have run
            (void)cudaGraphDestroy(graph);
            launches += per_step * replays * unroll;
            s += replays * unroll;                                     // what is left (< unroll steps, and the last, which wants phi) runs eagerly
        }
        const bool last = s + 1 == n_steps;
        t_launches = 0;
        rc = force_jerk_impl(n, xp, vp, n, xp, vp, m, eps2, a1, j1, last ? pot_out : nullptr, stream, true);
        if (rc != NB_OK) return rc;
        launches += t_launches;
        const int k = close_step(last);
        if (k < 0) return NB_ERR_CUDA;
        launches += k;
    }
    t_launches = launches;
    return NB_OK;
}

int nb_hermite4_block_step(int64_t n, float* x, float* v, const float* m, float* acc_io, float* jerk_io, double* t,
                           int64_t n_act, const int32_t* active, double t_now, float eps2, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || bad_count(n_act) || n_act > n) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2) || !std::isfinite(t_now)) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!x || !v || !m || !acc_io || !jerk_io || !t)) return NB_ERR_INVALID_VALUE;
    if (n_act > 0 && !active) return NB_ERR_INVALID_VALUE;
    if (3 * n > (int64_t)INT32_MAX) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_act == 0) return NB_OK;                                     // nobody is due: the state stays as it is
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    const size_t b3 = ((size_t)3 * n * sizeof(float) + 255) / 256 * 256;
    rc = ensure(&ws->hstate, &ws->hstate_bytes, 6 * b3, stream);      // xp, vp [n]; a1, j1, x_i, v_i [n_act <= n]
    if (rc != NB_OK) return rc;
    char* base = reinterpret_cast<char*>(ws->hstate);
    float* xp = reinterpret_cast<float*>(base);
    float* vp = reinterpret_cast<float*>(base + b3);
    float* a1 = reinterpret_cast<float*>(base + 2 * b3);
    float* j1 = reinterpret_cast<float*>(base + 3 * b3);
    float* xi = reinterpret_cast<float*>(base + 4 * b3);
    float* vi = reinterpret_cast<float*>(base + 5 * b3);
    rc = ensure(&ws->jp2, &ws->jp2_bytes, (size_t)n * 2 * sizeof(float4), stream);
    if (rc != NB_OK) return rc;
    const int threads = 256;
    const unsigned ablocks = (unsigned)((n_act + threads - 1) / threads);
    const unsigned jblocks = (unsigned)((n + threads - 1) / threads);
    nb::nb_block_predict_pack_kernel<<<jblocks + ablocks, threads, 0, stream>>>(
        x, v, acc_io, jerk_io, m, t, t_now, xp, vp, reinterpret_cast<float4*>(ws->jp2), (int)n, (int)jblocks, active,
        (int)n_act, xi, vi);
    NB_CUDA(cudaGetLastError());
    rc = force_jerk_impl(n_act, xi, vi, n, xp, vp, m, eps2, a1, j1, nullptr, stream, true);
    if (rc != NB_OK) return rc;
    nb::nb_block_correct_kernel<<<ablocks, threads, 0, stream>>>(x, v, acc_io, jerk_io, t, active, a1, j1, t_now, (int)n_act);
    NB_CUDA(cudaGetLastError());
    t_launches += 2;
    return NB_OK;
}

int nb_block_step_size(int64_t n, const float* a0, const float* j0, const float* a1, const float* j1, const float* h, float eta,
                       float* dt_out, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || !(eta > 0.0f) || !std::isfinite(eta)) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!a0 || !j0 || !a1 || !j1 || !h || !dt_out)) return NB_ERR_INVALID_VALUE;
    if (3 * n > (int64_t)INT32_MAX) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n == 0) return NB_OK;
    nb::nb_block_step_size_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(a0, j0, a1, j1, h, eta, dt_out, (int)n);
    NB_CUDA(cudaGetLastError());
    t_launches = 1;
    return NB_OK;
}

int nb_block_schedule(int64_t n, const double* t, const double* dt, double* t_next_out, int32_t* active_out,
                      int32_t* n_act_out, void* stream_) {
    t_launches = 0;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    if (bad_count(n) || !t_next_out || !n_act_out) return NB_ERR_INVALID_VALUE;
    if (n > 0 && (!t || !dt || !active_out)) return NB_ERR_INVALID_VALUE;
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    WsGuard guard(dev, stream);
    Workspace* ws = guard.ws;
    const int n_blocks = (int)((n + nb::kSchedTile - 1) / nb::kSchedTile);
    // scratch: [n_blocks] double CTA minima | [n_blocks] int CTA counts -> offsets
    rc = ensure(&ws->tiles, &ws->tiles_bytes, (size_t)(n_blocks + 1) * (sizeof(double) + sizeof(int)), stream);
    if (rc != NB_OK) return rc;
    double* block_min = reinterpret_cast<double*>(ws->tiles);
    int* counts = reinterpret_cast<int*>(block_min + n_blocks + 1);
    if (n_blocks > 0) {
        nb::nb_sched_min_kernel<<<n_blocks, nb::kSchedThreads, 0, stream>>>(t, dt, (int)n, block_min);
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    nb::nb_sched_final_min_kernel<<<1, 1024, 0, stream>>>(block_min, n_blocks, t_next_out);
    NB_CUDA(cudaGetLastError());
    if (n_blocks > 0) {
        nb::nb_sched_count_kernel<<<n_blocks, nb::kSchedThreads, 0, stream>>>(t, dt, (int)n, t_next_out, counts);
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    nb::nb_sched_scan_kernel<<<1, 1024, 0, stream>>>(counts, n_blocks, n_act_out);
    NB_CUDA(cudaGetLastError());
    if (n_blocks > 0) {
        nb::nb_sched_scatter_kernel<<<n_blocks, nb::kSchedThreads, 0, stream>>>(t, dt, (int)n, t_next_out, counts, active_out);
        NB_CUDA(cudaGetLastError());
        ++t_launches;
    }
    t_launches += 2;
    return NB_OK;
}

int nb_plan_query(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]) {
    if (!out || bad_count(n_i) || bad_count(n_j) || n_i < 1 || n_j < 1) return NB_ERR_INVALID_VALUE;
    const nb::Plan p = nb::make_plan(n_i, n_j, sm_count);
    out[0] = p.K; out[1] = p.WI; out[2] = p.WJ; out[3] = p.S;
    out[4] = p.tiles_i; out[5] = p.tile_i; out[6] = p.tile_j; out[7] = p.stages;
    return NB_OK;
}

int64_t nb_last_launch_count(void) { return t_launches; }

int nb_profile_enable(int on) {
    t_profile = (on != 0);
    return NB_OK;
}

int nb_profile_read(int64_t* n_launches, double* total_ms) {
    if (!n_launches || !total_ms) return NB_ERR_INVALID_VALUE;
    double sum = 0.0;
    int64_t n = 0;
    int rc = NB_OK;
    for (auto& ev : t_events) {
        float ms = 0.0f;
        cudaError_t e = cudaEventSynchronize(ev.second);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ev.first, ev.second);
        if (e != cudaSuccess) {
            t_last_cuda_error = (int)e;
            (void)cudaGetLastError();
            rc = NB_ERR_CUDA;
        } else {
            sum += ms;
            ++n;
        }
        (void)cudaEventDestroy(ev.first);
        (void)cudaEventDestroy(ev.second);
    }
    t_events.clear();
    *n_launches = n;
    *total_ms = sum;
    return rc;
}

int nb_release_workspace(void) {
    int dev = 0;
    NB_CUDA(cudaGetDevice(&dev));
    NB_CUDA(cudaDeviceSynchronize());
    std::lock_guard<std::mutex> lock(g_mutex);
    for (auto it = g_ws.begin(); it != g_ws.end();) {
        if (it->first.first == dev) {
            free_workspace(&it->second);
            it = g_ws.erase(it);
        } else {
            ++it;
        }
    }
    return NB_OK;
}

int nb_release_stream(void* stream_) {
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(stream_);
    int dev = 0;
    NB_CUDA(cudaGetDevice(&dev));
    NB_CUDA(cudaStreamSynchronize(stream));
    std::lock_guard<std::mutex> lock(g_mutex);
    auto it = g_ws.find(std::make_pair(dev, stream));
    if (it != g_ws.end()) {
        free_workspace(&it->second);
        g_ws.erase(it);
    }
    return NB_OK;
}

int nb_plan_query_small(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]) {
    if (!out || bad_count(n_i) || bad_count(n_j) || n_i < 1 || n_j < 1) return NB_ERR_INVALID_VALUE;
    const nb::SmallPlan p = nb::make_small_plan(n_i, n_j, sm_count);
    out[0] = p.NW; out[1] = p.KI; out[2] = p.LJ; out[3] = p.WJ; out[4] = p.S; out[5] = p.CS; out[6] = p.tiles_i;
    out[7] = nb::small_by_default(n_i, n_j) ? 1 : 0;
    return NB_OK;
}

int nb_plan_query_small_jerk(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]) {
    if (!out || bad_count(n_i) || bad_count(n_j) || n_i < 1 || n_j < 1) return NB_ERR_INVALID_VALUE;
    const nb::SmallPlan p = nb::make_small_jerk_plan(n_i, n_j, sm_count);
    out[0] = p.NW; out[1] = p.KI; out[2] = p.LJ; out[3] = p.WJ; out[4] = p.S; out[5] = p.CS; out[6] = p.tiles_i;
    out[7] = (nb::small_jerk_by_default(n_i, n_j, false) ? 1 : 0) | (nb::small_jerk_by_default(n_i, n_j, true) ? 2 : 0);
    return NB_OK;
}

int nb_debug_set(const char* key, const char* value) {
    if (!key) return NB_ERR_INVALID_VALUE;
    Knobs* fresh = new Knobs(knobs());                                 // copy, change, publish; the old copy is never freed
    if (!parse_knob(fresh, key, value)) {                              // (a test-only call: a few dozen bytes per change)
        delete fresh;
        return NB_ERR_INVALID_VALUE;
    }
    g_knobs.store(fresh, std::memory_order_release);
    return NB_OK;
}

int nb_debug_plan_exhaustive(int64_t n_i, int64_t n_j, int sm_count, int jerk, int64_t out[8]) {
    if (!out || bad_count(n_i) || bad_count(n_j) || n_i < 1 || n_j < 1) return NB_ERR_INVALID_VALUE;
    const nb::Plan p = jerk ? nb::make_plan_exhaustive(n_i, n_j, sm_count, 4, kHermiteInstPerPair, kHermitePartialBytes)
                            : nb::make_plan_exhaustive(n_i, n_j, sm_count);
    out[0] = p.K; out[1] = p.WI; out[2] = p.WJ; out[3] = p.S;
    out[4] = p.tiles_i; out[5] = p.tile_i; out[6] = jerk ? 256 : p.tile_j; out[7] = jerk ? ((p.WJ <= 2) ? 4 : 3) : p.stages;
    return NB_OK;
}

int64_t nb_debug_plans_computed(void) { return g_plans_computed.load(std::memory_order_relaxed); }

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// nb_force_noalloc (nbody_b200.h): the small-i-set kernel with the scratch of its j-split in a static device array.
// No cudaMalloc / cudaMallocAsync / cudaFree on this path, no Workspace, no events.
namespace {

constexpr size_t kNoAllocPartials = 131072;       // double4 entries: n_i * (S / CS) of a call must fit
constexpr size_t kNoAllocTickets = 4096;          // ints: tiles_i * CS <= (NB_NOALLOC_MAX_I / 8) * 8
constexpr size_t kNoAllocTicketOffset = kNoAllocPartials * sizeof(double4);
static_assert(kNoAllocTicketOffset + kNoAllocTickets * sizeof(int) == (size_t)NB_NOALLOC_SCRATCH_BYTES, "header and array agree");
static_assert((NB_NOALLOC_MAX_I / 8) * nb::kSmallClusterMax <= (int64_t)kNoAllocTickets, "one ticket per (i-tile, cluster rank)");
static_assert(kNoAllocPartials / NB_NOALLOC_MAX_I >= 1, "at least one group of partials at the largest n_i");

// One copy per GPU that loads the library, held until the process exits.  In HOST code this name is only a handle for
// cudaGetSymbolAddress -- never a device address: the kernel gets the pointer noalloc_scratch() resolves.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NB_NOALLOC_SCRATCH_BYTES];

std::atomic<unsigned char*> g_noalloc_ptr[64];     // per device ordinal (device_info rejects ordinals >= 64)

// Device address of the CURRENT device's copy; `dev` is the current device (device_info has just read it).
int noalloc_scratch(int dev, unsigned char** out) {
    unsigned char* p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
    if (!p) {                                      // once per device; two threads racing here resolve the same address
        void* q = nullptr;
        NB_CUDA(cudaGetSymbolAddress(&q, g_noalloc_scratch));
        if (!q) return NB_ERR_CUDA;
        p = static_cast<unsigned char*>(q);
        g_noalloc_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return NB_OK;
}

// The planner costs ~10 us per shape: repeated shapes are served from a fixed, direct-mapped table (no heap, unlike the
// std::map behind nb_force: this entry point allocates nothing on the host either).
nb::SmallPlan noalloc_plan(int64_t n_i, int64_t n_j, int sm_count) {
    struct Entry { int64_t key_i = -1, n_j = -1; int sm = 0; nb::SmallPlan plan{}; };
    static Entry table[64];
    static std::mutex table_mutex;
    const int64_t key_i = nb::small_plan_key_i(n_i);
    const size_t slot = (size_t)(((uint64_t)key_i * 0x9E3779B97F4A7C15ull) ^ ((uint64_t)n_j * 0xC2B2AE3D27D4EB4Full) ^ (uint64_t)sm_count) >> 58;
    {
        std::lock_guard<std::mutex> lock(table_mutex);
        const Entry& e = table[slot];
        if (e.key_i == key_i && e.n_j == n_j && e.sm == sm_count) return e.plan;
    }
    Entry fresh;
    fresh.key_i = key_i; fresh.n_j = n_j; fresh.sm = sm_count;
    fresh.plan = nb::make_small_plan(n_i, n_j, sm_count);              // outside the lock
    std::lock_guard<std::mutex> lock(table_mutex);
    table[slot] = fresh;
    return fresh.plan;
}

int force_noalloc_impl(int64_t n_i, const float* x_i, int64_t n_j, const float* x_j, const float* m_j, float eps2,
                       float* acc_out, float* pot_out, cudaStream_t stream) {
    if (bad_count(n_i) || bad_count(n_j)) return NB_ERR_INVALID_VALUE;
    if (!(eps2 >= 0.0f) || !std::isfinite(eps2)) return NB_ERR_INVALID_VALUE;
    if (n_i > 0 && (!x_i || !acc_out)) return NB_ERR_INVALID_VALUE;
    if (n_j > 0 && (!x_j || !m_j)) return NB_ERR_INVALID_VALUE;
    if (n_i > NB_NOALLOC_MAX_I) return NB_ERR_LIMIT;                   // before any CUDA call: nothing launched, nothing written
    int dev = 0;
    DeviceInfo info;
    int rc = device_info(&dev, &info);
    if (rc != NB_OK) return rc;
    if (n_i == 0) return NB_OK;
    if (n_j == 0) {
        NB_CUDA(cudaMemsetAsync(acc_out, 0, sizeof(float) * 3 * (size_t)n_i, stream));
        if (pot_out) NB_CUDA(cudaMemsetAsync(pot_out, 0, sizeof(float) * (size_t)n_i, stream));
        return NB_OK;
    }
    unsigned char* scratch = nullptr;
    rc = noalloc_scratch(dev, &scratch);
    if (rc != NB_OK) return rc;

    nb::SmallPlan sp = noalloc_plan(n_i, n_j, info.sm_count);
    const int64_t max_groups = (int64_t)(kNoAllocPartials / (size_t)n_i);   // >= 32 for n_i <= 4096
    if (sp.S / sp.CS > max_groups) sp.S = (int)(max_groups * sp.CS);   // fewer, longer j-chunks: the partials must fit
    const int n_groups = sp.S / sp.CS;
    if ((size_t)sp.tiles_i * sp.CS > kNoAllocTickets || (size_t)n_groups * (size_t)n_i > kNoAllocPartials) return NB_ERR_LIMIT;
    int* tickets = reinterpret_cast<int*>(scratch + kNoAllocTicketOffset);
    if (n_groups > 1)   // the array keeps the last call's contents: the counters this call takes tickets from start at zero
        NB_CUDA(cudaMemsetAsync(tickets, 0, sizeof(int) * (size_t)sp.tiles_i * sp.CS, stream));

    nb::SmallArgs sa;
    sa.x_i = x_i;
    sa.xj_raw = x_j;
    sa.mj_raw = m_j;
    sa.jp = nullptr;
    sa.acc = acc_out;
    sa.pot = pot_out;
    sa.partial = reinterpret_cast<double4*>(scratch);
    sa.tickets = tickets;
    sa.n_i = (int)n_i;
    sa.n_j = (int)n_j;
    sa.S = sp.S;
    sa.eps2 = eps2;
    sa.flag_offset = 0;
    // the mask modes of force_impl's small path (all three give the same bits)
    const int mode = (!pot_out && eps2 >= kUnmaskedMinEps2) ? nb::SMALL_NONE
                     : (eps2 >= kUnmaskedMinEps2 && nb::small_flag_pays(sp, n_j)) ? nb::SMALL_FLAG : nb::SMALL_EXACT;
    NB_CUDA(nb::small_launch(sp, sa, mode, stream));
    ++t_launches;
    return NB_OK;
}

}  // namespace

extern "C" {

int nb_force_noalloc(int64_t n_i, const float* x_i, int64_t n_j, const float* x_j, const float* m_j, float eps2,
                     float* acc_out, float* pot_out, void* stream) {
    t_launches = 0;
    return force_noalloc_impl(n_i, x_i, n_j, x_j, m_j, eps2, acc_out, pot_out, reinterpret_cast<cudaStream_t>(stream));
}

const char* nb_status_string(int status) {
    switch (status) {
        case NB_OK: return "NB_OK";
        case NB_ERR_INVALID_VALUE: return "NB_ERR_INVALID_VALUE: bad count, NULL required pointer, or eps2/dt out of range";
        case NB_ERR_CUDA: return "NB_ERR_CUDA: a CUDA runtime call failed (see nb_last_cuda_error)";
        case NB_ERR_ALLOC: return "NB_ERR_ALLOC: workspace allocation failed";
        case NB_ERR_UNSUPPORTED_DEVICE: return "NB_ERR_UNSUPPORTED_DEVICE: compute capability 10.x (B200, sm_100a) required";
        case NB_ERR_LIMIT: return "NB_ERR_LIMIT: nb_force_noalloc takes at most NB_NOALLOC_MAX_I = 4096 i-particles (its scratch is a fixed static device array)";
        default: return "unknown nb_status";
    }
}

int nb_last_cuda_error(void) { return t_last_cuda_error; }

int nb_version(void) { return NB_VERSION; }

}  // extern "C"
