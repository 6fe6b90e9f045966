/*
 * nb_pipeline.cuh -- the generalised pair kernel of the paper's section 4.5 ("CUNBODY-1 kernel"):
 * an arbitrary pair interaction given by three record widths and a "pipeline description", exactly the way the
 * paper's appendix drives its library (Fig. A.1 - A.4):
 *
 *     #define IDIM / JDIM / FDIM          floats per i-record, per j-record, per result record
 *     pipeline description                 INPUT_I[], INPUT_J[]  ->  OUTPUT[] += ...      (one (i, j) pair, FP32)
 *     cunbody_api(p_xj, p_xi, p_fi, ni, nj)     rows p_xj[nj][JDIM], p_xi[ni][IDIM], p_fi[ni][FDIM]
 *
 * A pipeline is a struct with  static constexpr int IDIM, JDIM, FDIM  and
 *     static __device__ void pair(const float* INPUT_I, const float* INPUT_J, float* OUTPUT);        // OUTPUT[] += ...
 * and  nb::pipeline_run<Pipeline>(p_xj, p_xi, p_fi, ni, nj, workspace, sm_count, stream)  is the cunbody_api call on
 * DEVICE rows.  That is all a user pipeline needs (the scalar path: `pipeline_kernel`).
 *
 * The fast path (`pipeline_kernel2`, taken when the pipeline also provides the PACKED hooks below) runs the pipeline the
 * way the library's own gravity kernels run theirs: two i-records per f32x2 instruction, K = 4 or 8 i-records per thread
 * in registers, j-records in double-buffered shared-memory tiles that the next tile's global loads overlap, Eq. (2)
 * two-level sums, and the coincident-pair rule decided per 128-j tile against a Bloom filter of the warp's i-positions
 * (nb_packed.cuh) instead of a select on every pair:
 *     static constexpr bool kPacked = true;
 *     static __device__ void prep_i(float* rec);                  // once per i-record at load (e.g. store -x canonicalised)
 *     template <bool MASKED>
 *     static __device__ void pair2(const u64* I2, const float* INPUT_J, u64* OUT2);   // I2[c] = (rec0[c], rec1[c]) packed
 *     static __device__ void finish(const double* sum, float* OUTPUT);               // FP64 totals -> result record
 *     static constexpr bool kCoincidentRule = true;                // records start with (x, y, z); equal positions add nothing:
 *                                                                  // MASKED = true is instantiated for the tiles that may hold one
 * Both paths: the j-range split over S CTAs with a fixed-order second pass (no floating-point atomics: bitwise
 * reproducible).
 *
 * libnbody_b200.so instantiates it for the paper's two listings, nb_cunbody_force (Fig. A.3) and nb_cunbody_force_jerk_pot
 * (Fig. A.4), and for a Lennard-Jones pipeline, see nbody_b200.h.  sm_100a, CUDA C++17, header only (needs nb_packed.cuh).
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <type_traits>

#include "nb_packed.cuh"

namespace nb {

constexpr int kPipeThreads = 256;    // threads per CTA
// i-records per thread: 4 for narrow records (Fig. A.3: +6 %), 2 for wide ones (Fig. A.4), by register budget
template <class P>
struct PipeK { static constexpr int value = (P::IDIM + 2 * P::FDIM <= 12) ? 4 : 2; };
constexpr int kPipeTile = 128;       // j-records per shared-memory tile
constexpr int kPipeBlock = 256;      // j-records per FP32 partial sum (Eq. (2))

template <class P>
__global__ void __launch_bounds__(kPipeThreads) pipeline_kernel(const float* __restrict__ p_xj, const float* __restrict__ p_xi,
                                                                float* __restrict__ p_fi, double* __restrict__ partial,
                                                                int n_i, int n_j, int S) {
    constexpr int I = P::IDIM, J = P::JDIM, F = P::FDIM, kPipeK = PipeK<P>::value;
    __shared__ float tile[kPipeTile * J];
    const int i0 = (blockIdx.x * kPipeThreads + threadIdx.x) * kPipeK;
    float xi[kPipeK][I];
#pragma unroll
    for (int k = 0; k < kPipeK; ++k) {
        const int i = min(i0 + k, n_i - 1);                            // clamped loads; stores are guarded
#pragma unroll
        for (int c = 0; c < I; ++c) xi[k][c] = p_xi[(size_t)i * I + c];
    }
    const int j_begin = (int)((long long)n_j * blockIdx.y / S);
    const int j_end = (int)((long long)n_j * (blockIdx.y + 1) / S);
    double run[kPipeK][F];
    float part[kPipeK][F];
#pragma unroll
    for (int k = 0; k < kPipeK; ++k)
#pragma unroll
        for (int c = 0; c < F; ++c) { run[k][c] = 0.0; part[k][c] = 0.0f; }
    int in_block = 0;
    for (int t0 = j_begin; t0 < j_end; t0 += kPipeTile) {
        const int nt = min(kPipeTile, j_end - t0);
        __syncthreads();                                               // previous tile fully read
        for (int q = threadIdx.x; q < nt * J; q += kPipeThreads) tile[q] = p_xj[(size_t)t0 * J + q];   // coalesced rows
        __syncthreads();
#pragma unroll 2
        for (int j = 0; j < nt; ++j) {
#pragma unroll
            for (int k = 0; k < kPipeK; ++k) P::pair(xi[k], &tile[j * J], part[k]);   // broadcast shared-memory reads
        }
        in_block += nt;
        if (in_block >= kPipeBlock || t0 + kPipeTile >= j_end) {       // partial -> running total, partial = 0
#pragma unroll
            for (int k = 0; k < kPipeK; ++k)
#pragma unroll
                for (int c = 0; c < F; ++c) { run[k][c] += (double)part[k][c]; part[k][c] = 0.0f; }
            in_block = 0;
        }
    }
#pragma unroll
    for (int k = 0; k < kPipeK; ++k) {
        const int i = i0 + k;
        if (i >= n_i) continue;
#pragma unroll
        for (int c = 0; c < F; ++c) {
            if (S == 1) p_fi[(size_t)i * F + c] = (float)run[k][c];
            else partial[((size_t)blockIdx.y * n_i + i) * F + c] = run[k][c];
        }
    }
}

template <int F>
__global__ void __launch_bounds__(128) pipeline_reduce_kernel(const double* __restrict__ partial, int n_i, int S,
                                                              float* __restrict__ p_fi) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_i) return;
    double s[F];
#pragma unroll
    for (int c = 0; c < F; ++c) s[c] = partial[(size_t)i * F + c];
    for (int q = 1; q < S; ++q)
#pragma unroll
        for (int c = 0; c < F; ++c) s[c] += partial[((size_t)q * n_i + i) * F + c];
#pragma unroll
    for (int c = 0; c < F; ++c) p_fi[(size_t)i * F + c] = (float)s[c];
}

// ---------------------------------------------------------------------------------------------------------------------
// The packed path.
template <class P, class = void> struct pipe_is_packed : std::false_type {};
template <class P> struct pipe_is_packed<P, std::enable_if_t<P::kPacked>> : std::true_type {};

// i-records per thread on the packed path: 8 (four packed pairs) for narrow records, 4 for wide ones, by register budget
template <class P>
struct PipeK2 { static constexpr int value = (P::IDIM + 3 * P::FDIM <= 17) ? 8 : 4; };
constexpr int kPipeTile2 = 128;      // j-records per tile = per Bloom test; two tiles per Eq. (2) block

template <class P>
__global__ void __launch_bounds__(kPipeThreads, 1) pipeline_kernel2(const float* __restrict__ p_xj, const float* __restrict__ p_xi,
                                                                   float* __restrict__ p_fi, double* __restrict__ partial,
                                                                   int n_i, int n_j, int S) {
    constexpr int I = P::IDIM, J = P::JDIM, F = P::FDIM, K = PipeK2<P>::value, K2 = K / 2;
    constexpr int TILE_FLOATS = kPipeTile2 * J, PRE = (TILE_FLOATS + kPipeThreads - 1) / kPipeThreads;
    extern __shared__ __align__(16) unsigned char pipe_smem[];
    float* tiles = reinterpret_cast<float*>(pipe_smem);                // [2][TILE_FLOATS]
    uint32_t* filt = reinterpret_cast<uint32_t*>(pipe_smem + 2 * TILE_FLOATS * sizeof(float)) + (threadIdx.x >> 5) * kBloomWords;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    // i-records: a warp owns 32 K consecutive records; pair k2 of a thread = records (2 k2) 32 + lane and (2 k2 + 1) 32 + lane
    const int i_base = (blockIdx.x * (kPipeThreads / 32) + warp) * (32 * K) + lane;
    u64 xi2[K2][I];
    if (P::kCoincidentRule) {
        uint32_t* all = reinterpret_cast<uint32_t*>(pipe_smem + 2 * TILE_FLOATS * sizeof(float));
        for (int q = threadIdx.x; q < (kPipeThreads / 32) * kBloomWords; q += kPipeThreads) all[q] = 0u;
        __syncthreads();
    }
#pragma unroll
    for (int k2 = 0; k2 < K2; ++k2) {
        float r0[I], r1[I];
        const int i0 = min(i_base + (2 * k2) * 32, n_i - 1), i1 = min(i_base + (2 * k2 + 1) * 32, n_i - 1);   // clamped loads
#pragma unroll
        for (int c = 0; c < I; ++c) { r0[c] = p_xi[(size_t)i0 * I + c]; r1[c] = p_xi[(size_t)i1 * I + c]; }
        if (P::kCoincidentRule) {
            bloom_set(filt, bloom_key(r0[0], r0[1], r0[2]));
            bloom_set(filt, bloom_key(r1[0], r1[1], r1[2]));
        }
        P::prep_i(r0); P::prep_i(r1);
#pragma unroll
        for (int c = 0; c < I; ++c) xi2[k2][c] = pack2(r0[c], r1[c]);
    }

    const int j_begin = (int)((long long)n_j * blockIdx.y / S);
    const int j_end = (int)((long long)n_j * (blockIdx.y + 1) / S);
    const int n_tiles = (j_end - j_begin + kPipeTile2 - 1) / kPipeTile2;
    double run[K][F];
    u64 part[K2][F];
#pragma unroll
    for (int k = 0; k < K; ++k)
#pragma unroll
        for (int c = 0; c < F; ++c) run[k][c] = 0.0;
#pragma unroll
    for (int k2 = 0; k2 < K2; ++k2)
#pragma unroll
        for (int c = 0; c < F; ++c) part[k2][c] = 0ull;

    // tile t: floats [j_begin + t T, ...) J, copied by the threads: loads of tile t + 1 are issued before tile t is swept
    float pre[PRE];
    auto load_tile = [&](int t) {
        const size_t base = (size_t)(j_begin + t * kPipeTile2) * J;
        const int nf = min(kPipeTile2, j_end - j_begin - t * kPipeTile2) * J;
#pragma unroll
        for (int u = 0; u < PRE; ++u) {
            const int q = threadIdx.x + u * kPipeThreads;
            pre[u] = (q < nf) ? p_xj[base + q] : 0.0f;
        }
    };
    auto store_tile = [&](int t) {
        float* dst = tiles + (t & 1) * TILE_FLOATS;
#pragma unroll
        for (int u = 0; u < PRE; ++u) {
            const int q = threadIdx.x + u * kPipeThreads;
            if (q < TILE_FLOATS) dst[q] = pre[u];
        }
    };
    if (n_tiles > 0) { load_tile(0); store_tile(0); }
    __syncthreads();                                                   // tile 0 staged, filters built
    for (int t = 0; t < n_tiles; ++t) {
        if (t + 1 < n_tiles) load_tile(t + 1);
        const float* tj = tiles + (t & 1) * TILE_FLOATS;
        const int nt = min(kPipeTile2, j_end - j_begin - t * kPipeTile2);
        bool masked = false;
        if (P::kCoincidentRule) {                                      // may a j of this tile coincide with an i of this warp?
            bool hit = false;
#pragma unroll
            for (int q = 0; q < kPipeTile2; q += 32) {
                const float* r = tj + min(q + lane, nt - 1) * J;
                hit |= bloom_test(filt, bloom_key(r[0], r[1], r[2]));
            }
            masked = __any_sync(0xffffffffu, hit);
        }
        if (masked) {
#pragma unroll 2
            for (int j = 0; j < nt; ++j)
#pragma unroll
                for (int k2 = 0; k2 < K2; ++k2) P::template pair2<true>(xi2[k2], tj + j * J, part[k2]);
        } else {
#pragma unroll 2
            for (int j = 0; j < nt; ++j)
#pragma unroll
                for (int k2 = 0; k2 < K2; ++k2) P::template pair2<false>(xi2[k2], tj + j * J, part[k2]);
        }
        if ((t & 1) || t + 1 == n_tiles) {                             // Eq. (2): partial -> running total every 256 j
#pragma unroll
            for (int k2 = 0; k2 < K2; ++k2)
#pragma unroll
                for (int c = 0; c < F; ++c) {
                    float lo, hi;
                    unpack2(part[k2][c], lo, hi);
                    run[2 * k2][c] += (double)lo; run[2 * k2 + 1][c] += (double)hi;
                    part[k2][c] = 0ull;
                }
        }
        if (t + 1 < n_tiles) store_tile(t + 1);                        // the other buffer: nobody reads it during tile t
        __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int i = i_base + k * 32;
        if (i >= n_i) continue;
        if (S == 1) {
            float out[F];
            P::finish(run[k], out);
#pragma unroll
            for (int c = 0; c < F; ++c) p_fi[(size_t)i * F + c] = out[c];
        } else {
#pragma unroll
            for (int c = 0; c < F; ++c) partial[((size_t)blockIdx.y * n_i + i) * F + c] = run[k][c];
        }
    }
}

template <class P>
__global__ void __launch_bounds__(128) pipeline_reduce_kernel2(const double* __restrict__ partial, int n_i, int S,
                                                               float* __restrict__ p_fi) {
    constexpr int F = P::FDIM;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_i) return;
    double s[F];
#pragma unroll
    for (int c = 0; c < F; ++c) s[c] = partial[(size_t)i * F + c];
    for (int q = 1; q < S; ++q)
#pragma unroll
        for (int c = 0; c < F; ++c) s[c] += partial[((size_t)q * n_i + i) * F + c];
    float out[F];
    P::finish(s, out);
#pragma unroll
    for (int c = 0; c < F; ++c) p_fi[(size_t)i * F + c] = out[c];
}

template <class P>
inline size_t pipeline_smem2() {
    return 2 * (size_t)kPipeTile2 * P::JDIM * sizeof(float) + (P::kCoincidentRule ? (size_t)(kPipeThreads / 32) * kBloomWords * sizeof(uint32_t) : 0);
}

// j-chunks across CTAs (a pure function of the sizes)
template <class P>
inline int pipeline_chunks(int64_t n_i, int64_t n_j, int sm_count) {
    if constexpr (pipe_is_packed<P>::value) {
        // one CTA of 8 warps per SM (registers): whole waves of sm_count CTAs, at least ~8 of them when the work allows
        constexpr int K = PipeK2<P>::value;
        const int64_t tiles = (n_i + kPipeThreads * K - 1) / (kPipeThreads * K);
        const int64_t s_max = n_j / (2 * kPipeTile2) > 0 ? n_j / (2 * kPipeTile2) : 1;
        int64_t best = 1;
        double best_eff = -1.0;
        for (int w = 1; w <= 24; ++w) {
            int64_t S = (int64_t)w * sm_count / tiles;
            if (S < 1) S = 1;
            if (S > s_max) S = s_max;
            if (S > 1024) S = 1024;
            const double ctas = double(tiles * S), waves = double((int64_t)((ctas + sm_count - 1) / sm_count));
            // wave quantisation x the start-up share of a CTA (~4 us of a CTA's life)
            const double work = double(n_i) * double(n_j) / (double(sm_count) * 9.0 * 2.0e9 / 1.0e6) / waves;   // us per wave at ~9 pairs/clk/SM
            const double eff = ctas / (waves * sm_count) * work / (work + 4.0);
            if (eff > best_eff * (1.0 + 1e-9)) { best_eff = eff; best = S; }
        }
        return (int)best;
    }
    constexpr int kPipeK = PipeK<P>::value;
    const int64_t tiles = (n_i + kPipeThreads * kPipeK - 1) / (kPipeThreads * kPipeK);
    int64_t S = (2 * (int64_t)sm_count + tiles - 1) / tiles;
    const int64_t s_max = n_j / kPipeBlock > 0 ? n_j / kPipeBlock : 1;
    if (S > s_max) S = s_max;
    if (S < 1) S = 1;
    if (S > 1024) S = 1024;
    return (int)S;
}

// Workspace bytes pipeline_run needs when pipeline_chunks(...) > 1 (caller-owned device memory).
template <class P>
inline size_t pipeline_workspace_bytes(int64_t n_i, int64_t n_j, int sm_count) {
    const int S = pipeline_chunks<P>(n_i, n_j, sm_count);
    return S > 1 ? (size_t)S * (size_t)n_i * P::FDIM * sizeof(double) : 0;
}

// The cunbody_api call on device rows.  Returns a cudaError_t.  n_j == 0 zero-fills p_fi.
template <class P>
inline cudaError_t pipeline_run(const float* p_xj, const float* p_xi, float* p_fi, int64_t n_i, int64_t n_j, void* workspace,
                                int sm_count, cudaStream_t stream) {
    if (n_i <= 0) return cudaSuccess;
    if (n_j <= 0) return cudaMemsetAsync(p_fi, 0, sizeof(float) * (size_t)n_i * P::FDIM, stream);
    const int S = pipeline_chunks<P>(n_i, n_j, sm_count);
    if (S > 1 && !workspace) return cudaErrorInvalidValue;
    if constexpr (pipe_is_packed<P>::value) {
        constexpr int K = PipeK2<P>::value;
        const size_t smem = pipeline_smem2<P>();
        static std::atomic<uint64_t> configured{0};                    // bit d: device d has the raised shared-memory limit
        int dev = 0;                                                   // (idempotent: a race only repeats the call)
        cudaError_t ce = cudaGetDevice(&dev);
        if (ce != cudaSuccess) return ce;
        const uint64_t bit = 1ull << (dev & 63);
        if (!(configured.load(std::memory_order_acquire) & bit)) {
            ce = cudaFuncSetAttribute(pipeline_kernel2<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (ce != cudaSuccess) return ce;
            configured.fetch_or(bit, std::memory_order_release);
        }
        const unsigned tiles = (unsigned)((n_i + kPipeThreads * K - 1) / (kPipeThreads * K));
        pipeline_kernel2<P><<<dim3(tiles, (unsigned)S, 1), kPipeThreads, smem, stream>>>(p_xj, p_xi, p_fi, reinterpret_cast<double*>(workspace),
                                                                                       (int)n_i, (int)n_j, S);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess || S == 1) return e;
        pipeline_reduce_kernel2<P><<<(unsigned)((n_i + 127) / 128), 128, 0, stream>>>(reinterpret_cast<const double*>(workspace),
                                                                                    (int)n_i, S, p_fi);
        return cudaGetLastError();
    } else {
        constexpr int kPipeK = PipeK<P>::value;
        const unsigned tiles = (unsigned)((n_i + kPipeThreads * kPipeK - 1) / (kPipeThreads * kPipeK));
        pipeline_kernel<P><<<dim3(tiles, (unsigned)S, 1), kPipeThreads, 0, stream>>>(p_xj, p_xi, p_fi, reinterpret_cast<double*>(workspace),
                                                                                   (int)n_i, (int)n_j, S);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess || S == 1) return e;
        pipeline_reduce_kernel<P::FDIM><<<(unsigned)((n_i + 127) / 128), 128, 0, stream>>>(reinterpret_cast<const double*>(workspace),
                                                                                         (int)n_i, S, p_fi);
        return cudaGetLastError();
    }
}

}  // namespace nb
