/*
 * nb_pipeline.cuh -- the generalised pair kernel of the paper's section 4.5 ("CUNBODY-1 kernel"):
 * an arbitrary pair interaction given by three record widths and a "pipeline description", exactly the way the
 * paper's appendix drives its library (Fig. A.1 - A.4):
 *
 *     #define IDIM / JDIM / FDIM          floats per i-record, per j-record, per result record
 *     pipeline description                 INPUT_I[], INPUT_J[]  ->  OUTPUT[] += ...      (one (i, j) pair, FP32)
 *     cunbody_api(p_xj, p_xi, p_fi, ni, nj)     rows p_xj[nj][JDIM], p_xi[ni][IDIM], p_fi[ni][FDIM]
 *
 * Here a pipeline is a struct with  static constexpr int IDIM, JDIM, FDIM  and
 *     static __device__ void pair(const float* INPUT_I, const float* INPUT_J, float* OUTPUT);   // OUTPUT[] += ...
 * and  nb::pipeline_run<Pipeline>(p_xj, p_xi, p_fi, ni, nj, stream)  is the cunbody_api call on DEVICE rows.
 * The scheme around the pipeline is the same as for the library's own gravity kernels: i-records stationary in
 * registers (2 or 4 per thread), j-records streamed through shared memory in tiles and read as warp broadcasts, Eq. (2)
 * two-level sums (FP32 partials over 256 j, FP64 running totals), the j-range split over S CTAs with a fixed-order
 * second pass (no floating-point atomics: bitwise reproducible).  The specialised kernels (packed FP32, TMA rings,
 * coincidence lists) are 1.8x faster for gravity; this header is for the interactions the library does not ship.
 *
 * libnbody_b200.so instantiates it for the paper's two listings: nb_cunbody_force (Fig. A.3) and
 * nb_cunbody_force_jerk_pot (Fig. A.4), see nbody_b200.h.  sm_100a, CUDA C++17, header only.
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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

// j-chunks across CTAs so that the grid fills the device about twice over (a pure function of the sizes)
template <class P>
inline int pipeline_chunks(int64_t n_i, int64_t n_j, int sm_count) {
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
    constexpr int kPipeK = PipeK<P>::value;
    const int S = pipeline_chunks<P>(n_i, n_j, sm_count);
    if (S > 1 && !workspace) return cudaErrorInvalidValue;
    const unsigned tiles = (unsigned)((n_i + kPipeThreads * kPipeK - 1) / (kPipeThreads * kPipeK));
    pipeline_kernel<P><<<dim3(tiles, (unsigned)S, 1), kPipeThreads, 0, stream>>>(p_xj, p_xi, p_fi, reinterpret_cast<double*>(workspace),
                                                                               (int)n_i, (int)n_j, S);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || S == 1) return e;
    pipeline_reduce_kernel<P::FDIM><<<(unsigned)((n_i + 127) / 128), 128, 0, stream>>>(reinterpret_cast<const double*>(workspace),
                                                                                     (int)n_i, S, p_fi);
    return cudaGetLastError();
}

}  // namespace nb
