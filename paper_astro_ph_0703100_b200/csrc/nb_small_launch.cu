// nb_small_launch.cu -- instantiations and launch dispatch of nb_small_kernel (nb_small.cuh), a translation unit of
// its own so that it compiles in parallel with nbody_b200.cu.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "nb_small.cuh"
#include "nb_plan.h"
#include "nb_small_launch.h"

namespace nb {

// dynamic shared memory: the staged j-pairs (reused for the reductions), then -- SMALL_FLAG -- the tile's Bloom filter and
// the slot bitmaps of marked pairs
size_t small_smem_bytes(const SmallPlan& p, int64_t n_j, bool flag, int* flag_offset) {
    const int Q = p.WJ * p.LJ;
    const int64_t chunk_max = (n_j + p.S - 1) / p.S + 2;     // as in nb_small_kernel (even chunk boundaries)
    const int round_max = (int)(chunk_max < kSmallRoundJ ? chunk_max : kSmallRoundJ);
    const int pstride = small_pair_stride(small_slot_len(round_max, Q));
    const size_t stage = (size_t)Q * pstride * 32;
    const size_t red = ((p.WJ > 1 ? (size_t)p.WJ * p.tile_i : 0) + (size_t)p.tile_i) * sizeof(double4);
    size_t bytes = ((stage > red ? stage : red) + 127) / 128 * 128;
    *flag_offset = (int)bytes;
    if (flag) bytes += (size_t)kBloomWords * sizeof(uint32_t) + (size_t)Q * small_flag_words(pstride) * sizeof(unsigned long long);
    return bytes + 128;
}

namespace {

template <int NW, int KI, int LJ, int WJ, int MODE, bool PHI, int CS>
cudaError_t launch_inst(const SmallPlan& p, const SmallArgs& a, size_t smem, cudaStream_t stream) {
    auto kern = nb_small_kernel<NW, KI, LJ, WJ, MODE, PHI, CS>;
    static std::atomic<uint64_t> configured{0};                       // bit d: device d has the raised shared-memory limit
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint64_t bit = 1ull << (dev & 63);
    if (!(configured.load(std::memory_order_acquire) & bit)) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
        if (e != cudaSuccess) return e;
        configured.fetch_or(bit, std::memory_order_release);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)p.tiles_i, (unsigned)p.S, 1);
    cfg.blockDim = dim3(32 * NW, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    // programmatic stream serialisation: the grid may be scheduled before the previous kernel of the stream has drained; the
    // kernel's first instruction is griddepcontrol.wait (a small call is ~2.4 us of launch around a few us of work)
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = p.pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (CS > 1) {
        attr[1].id = cudaLaunchAttributeClusterDimension;
        attr[1].val.clusterDim.x = 1;
        attr[1].val.clusterDim.y = (unsigned)p.CS;                    // 2, 4 or 8: the kernel reads the size from the hardware
        attr[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, kern, a);
}

template <int NW, int KI, int LJ, int WJ, int MODE, bool PHI>
cudaError_t launch_cs(const SmallPlan& p, const SmallArgs& a, size_t smem, cudaStream_t stream) {
    constexpr int TILE_I = (NW / WJ) * KI * (32 / LJ);
    if (p.CS == 1) return launch_inst<NW, KI, LJ, WJ, MODE, PHI, 1>(p, a, smem, stream);
    if constexpr (TILE_I % kSmallClusterMax == 0) {
        if (p.CS == 2 || p.CS == 4 || p.CS == kSmallClusterMax) return launch_inst<NW, KI, LJ, WJ, MODE, PHI, kSmallClusterMax>(p, a, smem, stream);
    }
    return cudaErrorInvalidValue;
}

template <int NW, int KI, int MODE, bool PHI>
cudaError_t launch_wide(const SmallPlan& p, const SmallArgs& a, size_t smem, cudaStream_t stream) {
    switch (p.WJ) {
        case 1: return launch_cs<NW, KI, 1, 1, MODE, PHI>(p, a, smem, stream);
        case 2: return launch_cs<NW, KI, 1, 2, MODE, PHI>(p, a, smem, stream);
        case 4: return launch_cs<NW, KI, 1, 4, MODE, PHI>(p, a, smem, stream);
        case 8: return launch_cs<NW, KI, 1, 8, MODE, PHI>(p, a, smem, stream);
        case 16:
            if constexpr (NW == 16) return launch_cs<NW, KI, 1, 16, MODE, PHI>(p, a, smem, stream);
            return cudaErrorInvalidValue;
        default: return cudaErrorInvalidValue;
    }
}

// the shapes of nb::small_shape_ok (nb_plan.h)
template <int MODE, bool PHI>
cudaError_t launch_shape(const SmallPlan& p, const SmallArgs& a, size_t smem, cudaStream_t stream) {
    if (!small_shape_ok(p.NW, p.KI, p.LJ, p.WJ, p.CS)) return cudaErrorInvalidValue;
    if (p.LJ == 2) return launch_cs<8, 1, 2, 8, MODE, PHI>(p, a, smem, stream);
    if (p.LJ == 4) return launch_cs<8, 1, 4, 8, MODE, PHI>(p, a, smem, stream);
    if (p.NW == 16) return p.KI == 2 ? launch_wide<16, 2, MODE, PHI>(p, a, smem, stream) : launch_wide<16, 1, MODE, PHI>(p, a, smem, stream);
    return p.KI == 2 ? launch_wide<8, 2, MODE, PHI>(p, a, smem, stream) : launch_wide<8, 1, MODE, PHI>(p, a, smem, stream);
}

cudaError_t launch_flag(const SmallPlan& p, const SmallArgs& a, size_t smem, cudaStream_t stream) {
    if (!small_shape_ok(p.NW, p.KI, p.LJ, p.WJ, p.CS) || p.LJ != 1) return cudaErrorInvalidValue;
    if (p.NW == 16) return p.KI == 2 ? launch_wide<16, 2, SMALL_FLAG, true>(p, a, smem, stream) : launch_wide<16, 1, SMALL_FLAG, true>(p, a, smem, stream);
    return p.KI == 2 ? launch_wide<8, 2, SMALL_FLAG, true>(p, a, smem, stream) : launch_wide<8, 1, SMALL_FLAG, true>(p, a, smem, stream);
}

}  // namespace

cudaError_t small_launch(const SmallPlan& p, SmallArgs a, int mode, cudaStream_t stream) {
    if (p.S % p.CS != 0 || p.S < 1) return cudaErrorInvalidValue;
    if (mode == SMALL_FLAG && p.LJ != 1) mode = SMALL_EXACT;           // the marked-pair branch needs a warp-uniform j-slot
    const size_t smem = small_smem_bytes(p, a.n_j, mode == SMALL_FLAG, &a.flag_offset);
    switch (mode) {
        case SMALL_NONE: return launch_shape<SMALL_NONE, false>(p, a, smem, stream);
        case SMALL_FLAG: return launch_flag(p, a, smem, stream);
        default: return launch_shape<SMALL_EXACT, true>(p, a, smem, stream);
    }
}

}  // namespace nb
