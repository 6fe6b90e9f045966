// nb_small_hermite_launch.cu -- instantiations and launch of nb_small_hermite_kernel (nb_small_hermite.cuh): a translation
// unit of its own, compiled side by side with the others (build.py).
#include "nb_small_hermite_launch.h"

#include <atomic>

#include "nb_plan.h"
#include "nb_small_hermite.cuh"

namespace nb {

size_t small_hermite_smem_bytes(const SmallPlan& p, int64_t n_j) {
    const int Q = p.WJ * p.LJ;
    const int64_t chunk_max = (n_j + p.S - 1) / p.S + 2;     // as in nb_small_hermite_kernel (even chunk boundaries)
    const int round_max = (int)(chunk_max < kSmallHRoundJ ? chunk_max : kSmallHRoundJ);
    const size_t stage = (size_t)Q * small_h_slot_stride(small_slot_len(round_max, Q)) * sizeof(float4);
    const size_t red = ((p.WJ > 1 ? (size_t)p.WJ * p.tile_i : 0) + 2 * (size_t)p.tile_i) * kHermiteAcc * sizeof(double);
    return ((stage > red ? stage : red) + 127) / 128 * 128 + 128;
}

namespace {

template <int NW, int LJ, int WJ, bool PHI, int CS>
cudaError_t launch_inst(const SmallPlan& p, const SmallHermiteArgs& a, size_t smem, cudaStream_t stream) {
    auto kern = nb_small_hermite_kernel<NW, LJ, WJ, PHI, CS>;
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
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // the kernel's first instruction is griddepcontrol.wait
    attr[0].val.programmaticStreamSerializationAllowed = p.pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (CS > 1) {
        attr[1].id = cudaLaunchAttributeClusterDimension;
        attr[1].val.clusterDim.x = 1;
        attr[1].val.clusterDim.y = (unsigned)p.CS;                     // 2, 4 or 8: the kernel reads the size from the hardware
        attr[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, kern, a);
}

template <int NW, int LJ, int WJ, bool PHI>
cudaError_t launch_cs(const SmallPlan& p, const SmallHermiteArgs& a, size_t smem, cudaStream_t stream) {
    if (p.CS == 1) return launch_inst<NW, LJ, WJ, PHI, 1>(p, a, smem, stream);
    if (p.CS == 2 || p.CS == 4 || p.CS == kSmallClusterMax) return launch_inst<NW, LJ, WJ, PHI, kSmallClusterMax>(p, a, smem, stream);
    return cudaErrorInvalidValue;
}

template <bool PHI>
cudaError_t launch_shape(const SmallPlan& p, const SmallHermiteArgs& a, size_t smem, cudaStream_t stream) {
    if (p.NW == 8 && p.LJ == 2 && p.WJ == 8) return launch_cs<8, 2, 8, PHI>(p, a, smem, stream);
    if (p.NW == 8 && p.LJ == 4 && p.WJ == 8) return launch_cs<8, 4, 8, PHI>(p, a, smem, stream);
    if (p.NW != 16 || p.LJ != 1) return cudaErrorInvalidValue;
    switch (p.WJ) {
        case 2: return launch_cs<16, 1, 2, PHI>(p, a, smem, stream);
        case 4: return launch_cs<16, 1, 4, PHI>(p, a, smem, stream);
        case 8: return launch_cs<16, 1, 8, PHI>(p, a, smem, stream);
        case 16: return launch_cs<16, 1, 16, PHI>(p, a, smem, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t small_hermite_launch(const SmallPlan& p, const SmallHermiteArgs& a, cudaStream_t stream) {
    if (!small_jerk_shape_ok(p.NW, p.LJ, p.WJ, p.CS) || p.KI != 1 || p.S % p.CS != 0 || p.S < 1) return cudaErrorInvalidValue;
    const size_t smem = small_hermite_smem_bytes(p, a.n_j);
    return a.pot ? launch_shape<true>(p, a, smem, stream) : launch_shape<false>(p, a, smem, stream);
}

}  // namespace nb
