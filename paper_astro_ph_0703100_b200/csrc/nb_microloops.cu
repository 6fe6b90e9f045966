// nb_microloops.cu -- the measurements behind the "alu" roofline of DESIGN.md section 6 and the small-call planner's
// efficiency table (nb_plan.h: small_loop_eff), as a stand-alone program for one B200:
//   * unit rates: FFMA, FFMA2, MUFU.RSQ, FADD2 with a scalar broadcast operand, FFMA2 with three distinct register pairs
//     (warp instructions per clock per SM) -- SURVEY.md section 8.3.3 asks for them before any fraction is quoted;
//   * the pair-interaction loop bodies fed from shared memory as in the kernels: packed over i (nb_kernels.cuh) and packed
//     over j (nb_small.cuh), with and without the exact coincidence mask, by warps per SM -- as a fraction of the
//     13-instruction FP32 roofline (128 lanes / 13 instructions per clock per SM).
// Build and run:  python -m paper_astro_ph_0703100_b200.build --microloops && ./paper_astro_ph_0703100_b200/nb_microloops
//   * `nb_microloops --phases`: nb_small_kernel on a C2-shaped call (512 x 65536) with a time stamp after every phase
//     (staging, loop, lane / warp sums, ticket, final sums), per CTA: where a small call spends its time.
// Output of the round-2 runs: profiles/r02_microloops.md, profiles/r02_small_calls.md.
#define NB_SMALL_STAMPS   // this program only: nb_small_kernel writes %globaltimer / clock64 stamps of its phases
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <vector>
#include <algorithm>
#include <random>
#include <cstring>
#include "../../include/nb_packed.cuh"
#include "nb_small.cuh"
using namespace nb;

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1); } } while (0)

// ---------------- unit rates: N independent chains per thread
template <int MODE>   // 0 FFMA, 1 FFMA2, 2 MUFU.RSQ, 3 FADD2 with scalar operand, 4 FFMA2 3 distinct pairs
__global__ void unit_kernel(float* out, int iters, float seed) {
    float a[8]; u64 p[8];
    for (int k = 0; k < 8; ++k) { a[k] = seed + k + threadIdx.x; p[k] = pack2(a[k], a[k] + 1.f); }
    const float b = seed * 0.5f, c = seed * 0.25f;
    const u64 pb = pack2(b, b + 1.f), pc = pack2(c, c + 2.f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (MODE == 0) a[k] = fmaf(a[k], b, c);
            if (MODE == 1) p[k] = fma2(p[k], pb, pc);
            if (MODE == 2) a[k] = rsqrt_approx(a[k]);
            if (MODE == 3) p[k] = add2(p[k], pack2(b, b));
            if (MODE == 4) p[k] = fma2(pb, pc, p[k]);
        }
    }
    float s = 0; for (int k = 0; k < 8; ++k) { float lo, hi; unpack2(p[k], lo, hi); s += a[k] + lo + hi; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---------------- loop bodies from shared memory
// i-packed (nb_kernels.cuh pair_body): K/2 packed i-pairs per thread, one LDS.128 per j
template <int K, int MASK>
__global__ void ipacked_kernel(const float4* jp, int n_j, float* out, float eps2) {
    extern __shared__ float4 sj[];
    for (int q = threadIdx.x; q < n_j; q += blockDim.x) sj[q] = jp[q];
    __syncthreads();
    u64 nx[K / 2], ny[K / 2], nz[K / 2], ax[K / 2], ay[K / 2], az[K / 2], ph[K / 2];
    for (int k = 0; k < K / 2; ++k) {
        const float f = 0.001f * (threadIdx.x + 64 * k + blockIdx.x);
        nx[k] = pack2(f, f + 1.f); ny[k] = pack2(f * 2, f * 3); nz[k] = pack2(-f, f - 2.f);
        ax[k] = ay[k] = az[k] = ph[k] = 0ull;
    }
    const u64 e2 = pack2(eps2, eps2);
#pragma unroll 4
    for (int j = 0; j < n_j; ++j) {
        const float4 J = sj[j];
        const u64 xj = pack2(J.x, J.x), yj = pack2(J.y, J.y), zj = pack2(J.z, J.z), mj = pack2(J.w, J.w);
#pragma unroll
        for (int k = 0; k < K / 2; ++k) {
            const u64 dx = add2(xj, nx[k]), dy = add2(yj, ny[k]), dz = add2(zj, nz[k]);
            u64 r2 = fma2(dx, dx, e2); r2 = fma2(dy, dy, r2); r2 = fma2(dz, dz, r2);
            float ra, rb; unpack2(r2, ra, rb);
            if (MASK == MASK_EXACT) {
                float a0, a1, b0, b1, c0, c1; unpack2(dx, a0, a1); unpack2(dy, b0, b1); unpack2(dz, c0, c1);
                const uint32_t ta = __float_as_uint(a0) | __float_as_uint(b0) | __float_as_uint(c0);
                const uint32_t tb = __float_as_uint(a1) | __float_as_uint(b1) | __float_as_uint(c1);
                ra = ta == 0u ? __int_as_float(0x7f800000) : ra; rb = tb == 0u ? __int_as_float(0x7f800000) : rb;
            }
            const u64 u = pack2(rsqrt_approx(ra), rsqrt_approx(rb));
            const u64 u2 = mul2(u, u), mu = mul2(mj, u), mu3 = mul2(mu, u2);
            ax[k] = fma2(mu3, dx, ax[k]); ay[k] = fma2(mu3, dy, ay[k]); az[k] = fma2(mu3, dz, az[k]); ph[k] = add2(ph[k], mu);
        }
    }
    float s = 0;
    for (int k = 0; k < K / 2; ++k) { float lo, hi; unpack2(ax[k], lo, hi); s += lo + hi; unpack2(ay[k], lo, hi); s += lo + hi; unpack2(az[k], lo, hi); s += lo + hi; unpack2(ph[k], lo, hi); s += lo + hi; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// j-packed (nb_small.cuh pair_body_j2): KI i-particles per thread, two LDS.128 per j-pair; UNR = pairs unrolled
template <int KI, int MASK, int UNR>
__global__ void jpacked_kernel(const float4* jp2, int n_pairs, float* out, float eps2) {
    extern __shared__ float4 sj[];
    for (int q = threadIdx.x; q < 2 * n_pairs; q += blockDim.x) sj[q] = jp2[q];
    __syncthreads();
    u64 nx[KI], ny[KI], nz[KI], ax[KI], ay[KI], az[KI], ph[KI];
    for (int k = 0; k < KI; ++k) {
        const float f = 0.001f * (threadIdx.x + 64 * k + blockIdx.x);
        nx[k] = pack2(f, f); ny[k] = pack2(f * 2, f * 2); nz[k] = pack2(-f, -f);
        ax[k] = ay[k] = az[k] = ph[k] = 0ull;
    }
    const u64 e2 = pack2(eps2, eps2);
#pragma unroll UNR
    for (int p = 0; p < n_pairs; ++p) {
        const float4 A = sj[2 * p], B = sj[2 * p + 1];
        const u64 xj2 = pack2(A.x, A.y), yj2 = pack2(A.z, A.w), zj2 = pack2(B.x, B.y), mj2 = pack2(B.z, B.w);
#pragma unroll
        for (int k = 0; k < KI; ++k) pair_body_j2<MASK, true>(xj2, yj2, zj2, mj2, nx[k], ny[k], nz[k], e2, ax[k], ay[k], az[k], ph[k]);
    }
    float s = 0;
    for (int k = 0; k < KI; ++k) { float lo, hi; unpack2(ax[k], lo, hi); s += lo + hi; unpack2(ay[k], lo, hi); s += lo + hi; unpack2(az[k], lo, hi); s += lo + hi; unpack2(ph[k], lo, hi); s += lo + hi; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

static int g_sm = 148; static double g_hz = 1.965e9;

// ---------------- phases of nb_small_kernel (--phases)
__global__ void marker_kernel(long long* t) { long long v; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(v)); *t = v; }

template <int NW, int KI, int LJ, int WJ, int MODE, bool PHI>
void phase_run(const char* name, int n_i, int n_j, int S, float* xi, float* xj, float* mj, float* acc, float* pot, double4* partial, int* tickets, long long* stamps,
               void* flush, size_t flush_bytes) {
    constexpr int TILE = (NW / WJ) * KI * (32 / LJ);
    const int tiles = (n_i + TILE - 1) / TILE, Q = WJ * LJ;
    const int chunk_max = (n_j + S - 1) / S + 2, round_max = chunk_max < kSmallRoundJ ? chunk_max : kSmallRoundJ;
    const int pstride = small_pair_stride(small_slot_len(round_max, Q));
    size_t stage = (size_t)Q * pstride * 32, red = ((WJ > 1 ? (size_t)WJ * TILE : 0) + TILE) * 32;
    size_t smem = ((stage > red ? stage : red) + 127) / 128 * 128;
    SmallArgs a{}; a.x_i = xi; a.xj_raw = xj; a.mj_raw = mj; a.jp = nullptr; a.acc = acc; a.pot = PHI ? pot : nullptr; a.partial = partial; a.tickets = tickets;
    a.n_i = n_i; a.n_j = n_j; a.S = S; a.eps2 = 1.f / 16384; a.stamps = nullptr;
    a.flag_offset = (int)smem;
    if (MODE == SMALL_FLAG) smem += (size_t)kBloomWords * 4 + (size_t)Q * small_flag_words(pstride) * 8;
    smem += 128;
    auto kern = nb_small_kernel<NW, KI, LJ, WJ, MODE, PHI, 1>;
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024));
    const int n_ctas = tiles * S;
    for (int r = 0; r < 5; ++r) kern<<<dim3(tiles, S), 32 * NW, smem>>>(a);
    CK(cudaDeviceSynchronize());
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    CK(cudaEventRecord(e0)); for (int r = 0; r < 20; ++r) kern<<<dim3(tiles, S), 32 * NW, smem>>>(a); CK(cudaEventRecord(e1)); CK(cudaEventSynchronize(e1));
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
    printf("%s: grid %d x %d, %d threads, smem %zu: %.2f us per back-to-back launch\n", name, tiles, S, 32 * NW, smem, ms * 1e3 / 20);
    a.stamps = stamps;
    long long* mark = stamps + 4096 * 16 - 8;
    // warm: the stamped launch follows 20 identical ones; cold: it follows a write of flush_bytes (> L2) -- inputs, code
    // and the workspace then come from DRAM.  A one-thread marker kernel in front gives the launch gap.
    for (int cold = 0; cold < 2; ++cold) {
        std::vector<double> first(7, 0.0), last(7, 0.0), own(7, 0.0); double gap = 0; int reps = 5; std::vector<size_t> cnt(7, 0);
        for (int r = 0; r < reps; ++r) {
            CK(cudaMemset(stamps, 0, (size_t)4096 * 16 * 8));
            if (cold) CK(cudaMemsetAsync(flush, r + 1, flush_bytes));
            marker_kernel<<<1, 1>>>(mark);
            kern<<<dim3(tiles, S), 32 * NW, smem>>>(a); CK(cudaDeviceSynchronize());
            std::vector<long long> h(4096 * 16); CK(cudaMemcpy(h.data(), stamps, h.size() * 8, cudaMemcpyDeviceToHost));
            long long t0 = h[0]; for (int c = 0; c < n_ctas; ++c) t0 = std::min(t0, h[c * 16]);
            gap += (t0 - h[4096 * 16 - 8]) * 1e-3 / reps;
            for (int k = 0; k < 7; ++k) {
                std::vector<double> g, c;
                for (int q = 0; q < n_ctas; ++q) if (h[q * 16 + k]) { g.push_back((h[q * 16 + k] - t0) * 1e-3); c.push_back((h[q * 16 + 8 + k] - h[q * 16 + 8]) / 1.965e3); }
                if (g.empty()) continue;
                std::sort(g.begin(), g.end()); std::sort(c.begin(), c.end());
                first[k] += g.front() / reps; last[k] += g.back() / reps; own[k] += c[c.size() / 2] / reps; cnt[k] = g.size();
            }
        }
        const char* ph[7] = {"start", "staged", "loop done", "tile sums out", "ticket taken", "final sums done", "after sleep"};
        printf("  %s (mean of %d launches): first CTA starts %.2f us after the marker kernel's stamp\n", cold ? "COLD, after a 256 MiB write" : "WARM", reps, gap);
        for (int k = 0; k < 7; ++k) if (cnt[k])
            printf("   %-16s (%3zu CTAs)  since first CTA start [us]: first %.2f last %.2f | since own start (clock64 at 1.965 GHz), median CTA [us]: %.2f\n",
                   ph[k], cnt[k], first[k], last[k], own[k]);
    }
}

static int phases_main() {
    const int n_i = 512, n_j = 65536;
    std::mt19937 rng(1); std::normal_distribution<float> nd;
    std::vector<float> hx(3 * n_j), hm(n_j, 1.f / n_j), hi(3 * n_i);
    for (auto& v : hx) v = nd(rng);
    for (int i = 0; i < n_i; ++i) for (int c = 0; c < 3; ++c) hi[3 * i + c] = hx[3 * (i * 97) + c];
    float *xi, *xj, *mj, *acc, *pot; double4* partial; int* tickets; long long* stamps;
    CK(cudaMalloc(&xi, hi.size() * 4)); CK(cudaMalloc(&xj, hx.size() * 4)); CK(cudaMalloc(&mj, hm.size() * 4)); CK(cudaMalloc(&acc, n_i * 12)); CK(cudaMalloc(&pot, n_i * 4));
    CK(cudaMalloc(&partial, (size_t)512 * n_i * 32)); CK(cudaMalloc(&tickets, 4096)); CK(cudaMemset(tickets, 0, 4096)); CK(cudaMalloc(&stamps, 4096 * 16 * 8));
    CK(cudaMemcpy(xi, hi.data(), hi.size() * 4, cudaMemcpyHostToDevice)); CK(cudaMemcpy(xj, hx.data(), hx.size() * 4, cudaMemcpyHostToDevice)); CK(cudaMemcpy(mj, hm.data(), hm.size() * 4, cudaMemcpyHostToDevice));
    void* flush; const size_t flush_bytes = 256u << 20; CK(cudaMalloc(&flush, flush_bytes));
#define PH(NW, KI, LJ, WJ, MODE, PHI, name, ni, nj, S) phase_run<NW, KI, LJ, WJ, MODE, PHI>(name, ni, nj, S, xi, xj, mj, acc, pot, partial, tickets, stamps, flush, flush_bytes)
    PH(16, 2, 1, 8, SMALL_EXACT, true, "C2 512 x 65536 NW16 KI2 WJ8 exact S37", n_i, n_j, 37);
    PH(16, 2, 1, 16, SMALL_EXACT, true, "C2 512 x 65536 NW16 KI2 WJ16 exact S18", n_i, n_j, 18);
    PH(16, 2, 1, 16, SMALL_FLAG, true, "C2 512 x 65536 NW16 KI2 WJ16 flag S18 (the library's plan)", n_i, n_j, 18);
    PH(16, 1, 1, 8, SMALL_EXACT, true, "C2 512 x 65536 NW16 KI1 WJ8 exact S18", n_i, n_j, 18);
    PH(16, 2, 1, 16, SMALL_NONE, false, "C2 512 x 65536 NW16 KI2 WJ16 no mask, no phi S18", n_i, n_j, 18);
    PH(16, 1, 1, 8, SMALL_EXACT, true, "C0-shaped 512 x 2048 of the same arrays, NW16 KI1 WJ8 exact S4", 512, 2048, 4);
    PH(8, 1, 4, 8, SMALL_EXACT, true, "1 x 2, NW8 KI1 LJ4 WJ8 exact S1 (launch floor)", 1, 2, 1);
        return 0;
}

template <class F> static double run(F f, int reps = 20) {
    cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    for (int r = 0; r < 3; ++r) f();
    CK(cudaDeviceSynchronize());
    CK(cudaEventRecord(e0));
    for (int r = 0; r < reps; ++r) f();
    CK(cudaEventRecord(e1)); CK(cudaEventSynchronize(e1));
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1)); CK(cudaGetLastError());
    return ms / reps * 1e-3;
}

int main(int argc, char** argv) {
    if (argc > 1 && !std::strcmp(argv[1], "--phases")) return phases_main();
    cudaDeviceProp prop; CK(cudaGetDeviceProperties(&prop, 0)); g_sm = prop.multiProcessorCount;
    int khz = 0; CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0)); g_hz = khz * 1e3;
    printf("# %s, %d SMs, clock attribute %.0f MHz (rates below are per SM per clock at that clock)\n", prop.name, g_sm, g_hz / 1e6);
    float* out; CK(cudaMalloc(&out, 64 << 20));
    const int n_j = 4096;
    std::vector<float4> h(2 * n_j);
    for (int q = 0; q < 2 * n_j; ++q) h[q] = make_float4(0.37f * q, 1.0f + 0.11f * q, -0.5f * q, 1.0f / n_j);
    float4* jp; CK(cudaMalloc(&jp, h.size() * sizeof(float4))); CK(cudaMemcpy(jp, h.data(), h.size() * sizeof(float4), cudaMemcpyHostToDevice));

    // ---- unit rates
    const int iters = 4096;
    const char* names[5] = {"FFMA (scalar, 3 registers)", "FFMA2 (2 register pairs + 1)", "MUFU.RSQ", "FADD2 (pair + scalar broadcast)", "FFMA2 (3 distinct pairs)"};
    for (int mode = 0; mode < 5; ++mode) {
        for (int warps : {4, 8, 16, 32}) {
            auto f = [&]() {
                switch (mode) {
                    case 0: unit_kernel<0><<<g_sm, 32 * warps>>>(out, iters, 1.5f); break;
                    case 1: unit_kernel<1><<<g_sm, 32 * warps>>>(out, iters, 1.5f); break;
                    case 2: unit_kernel<2><<<g_sm, 32 * warps>>>(out, iters, 1.5f); break;
                    case 3: unit_kernel<3><<<g_sm, 32 * warps>>>(out, iters, 1.5f); break;
                    default: unit_kernel<4><<<g_sm, 32 * warps>>>(out, iters, 1.5f); break;
                }
            };
            const double t = run(f);
            const double winst = double(iters) * 8 * warps;            // warp instructions per SM
            printf("unit | %-32s | %2d warps/SM | %.3f warp-inst/clk/SM\n", names[mode], warps, winst / (t * g_hz));
        }
    }

    // ---- loop bodies: fraction of the 13-instruction roofline (128 lanes / 13 pairs per clock per SM)
    const double roof = 128.0 / 13.0;
    CK(cudaFuncSetAttribute(ipacked_kernel<8, MASK_NONE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 << 10));
#define IP(K, M) { for (int warps : {8, 16}) { if (K == 8 && warps > 8) continue; \
        CK(cudaFuncSetAttribute(ipacked_kernel<K, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 << 10)); \
        auto f = [&]() { ipacked_kernel<K, M><<<g_sm, 32 * warps, n_j * 16>>>(jp, n_j, out, 1e-4f); }; \
        const double t = run(f); const double pairs = double(n_j) * K * 32 * warps; \
        printf("body | i-packed K=%d %-5s | %2d warps/SM | %.3f pairs/clk/SM = %.1f %% of roofline\n", K, M == MASK_NONE ? "plain" : "exact", warps, pairs / (t * g_hz), 100 * pairs / (t * g_hz) / roof); } }
    IP(8, MASK_NONE) IP(8, MASK_EXACT) IP(4, MASK_NONE) IP(4, MASK_EXACT) IP(2, MASK_NONE) IP(2, MASK_EXACT)
#define JP(KI, M, U) { for (int warps : {8, 16, 32}) { if (KI == 4 && warps > 16) continue; \
        CK(cudaFuncSetAttribute(jpacked_kernel<KI, M, U>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 << 10)); \
        auto f = [&]() { jpacked_kernel<KI, M, U><<<g_sm, 32 * warps, n_j * 16>>>(jp, n_j / 2, out, 1e-4f); }; \
        const double t = run(f); const double pairs = double(n_j) * KI * 32 * warps; \
        printf("body | j-packed KI=%d %-5s unroll %d | %2d warps/SM | %.3f pairs/clk/SM = %.1f %% of roofline\n", KI, M == MASK_NONE ? "plain" : "exact", U, warps, pairs / (t * g_hz), 100 * pairs / (t * g_hz) / roof); } }
    JP(4, MASK_NONE, 2) JP(4, MASK_EXACT, 2) JP(4, MASK_NONE, 1) JP(4, MASK_EXACT, 1)
    JP(2, MASK_NONE, 4) JP(2, MASK_EXACT, 4) JP(2, MASK_NONE, 2) JP(2, MASK_EXACT, 2)
    JP(1, MASK_NONE, 8) JP(1, MASK_EXACT, 8) JP(1, MASK_NONE, 4) JP(1, MASK_EXACT, 4)
    return 0;
}
