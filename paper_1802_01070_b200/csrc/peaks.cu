// peaks.cu -- microbenchmarks for the roofline denominators MEASURED_PEAKS.json lacks:
// plain FP64 FMA rate (bounds K1), L2-resident random 4-byte gathers, red.global.add.f32 / .v2.f32 into an
// L2-resident array (bound the direct projection path), shared-memory integer atomics and loads (bound the
// windowed projection path).  Each figure is the best of three timed launches after a warm-up, CUDA events.
#include <cstdio>

#include "pct_internal.cuh"

namespace pct {

constexpr int PK_THREADS = 256;

__device__ __forceinline__ unsigned lcg(unsigned s) { return s * 1664525u + 1013904223u; }

__global__ void __launch_bounds__(PK_THREADS) k_peak_fp64(double* out, int iters, double a, double b) {
    double r[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) r[k] = (double)(threadIdx.x + k);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) r[k] = fma(r[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += r[k];
    if (s == 12345.678) out[0] = s;          // never true; keeps the chain alive
}

// random 4-byte loads over `n` floats (n a power of two); 8 independent loads in flight per thread
__global__ void __launch_bounds__(PK_THREADS) k_peak_gather(const float* __restrict__ x, unsigned mask, int iters, float* out) {
    unsigned s = (blockIdx.x * PK_THREADS + threadIdx.x) * 2654435761u + 12345u;
    float acc = 0.f;
    for (int i = 0; i < iters; ++i) {
        unsigned idx[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) { s = lcg(s); idx[k] = (s >> 4) & mask; }
#pragma unroll
        for (int k = 0; k < 8; ++k) acc += __ldg(x + idx[k]);
    }
    if (acc == 12345.678f) out[0] = acc;
}

// mode 0: random addresses, scalar f32;  1: random, v2.f32 on float2 slots;  2: warp-contiguous (lane l -> base+l), v2
__global__ void __launch_bounds__(PK_THREADS) k_peak_red(float* __restrict__ d, unsigned mask, int iters, int mode) {
    unsigned s = (blockIdx.x * PK_THREADS + threadIdx.x) * 2654435761u + 999u;
    const unsigned lane = threadIdx.x & 31u;
    for (int i = 0; i < iters; ++i) {
        s = lcg(s);
        unsigned idx = (s >> 4) & mask;
        if (mode == 2) idx = ((__shfl_sync(0xffffffffu, idx, 0) & ~31u) + lane) & mask;
        if (mode == 0) asm volatile("red.global.add.f32 [%0], %1;" ::"l"(d + idx), "f"(1.0f) : "memory");
        else asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(reinterpret_cast<float2*>(d) + idx), "f"(1.0f), "f"(1.0f) : "memory");
    }
}

// shared-memory integer atomics (mode 0, 2) or loads (mode 1, 3) on `slots` 4-byte slots; modes 0/1: random addresses,
// modes 2/3: conflict-free (a random row of 32 slots per warp, lane l -> bank l)
__global__ void __launch_bounds__(1024) k_peak_smem(int slots_mask, int iters, int mode, int* out) {
    extern __shared__ int sm[];
    for (int i = threadIdx.x; i <= slots_mask; i += blockDim.x) sm[i] = 0;
    __syncthreads();
    // modes 2/3: the sequence depends on the warp only, so all lanes draw the same row and differ in the bank
    unsigned s = (mode >= 2 ? (blockIdx.x * blockDim.x + threadIdx.x) >> 5 : blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 77u;
    const int lane_or = mode >= 2 ? (int)(threadIdx.x & 31u) : 0, row_mask = mode >= 2 ? slots_mask & ~31 : slots_mask;
    int acc = 0;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            s = lcg(s);
            const int idx = (int)((s >> 8) & (unsigned)row_mask) | lane_or;
            if ((mode & 1) == 0) atomicAdd(&sm[idx], 1); else acc += sm[idx];
        }
    }
    __syncthreads();
    if (acc == 123456789 || sm[threadIdx.x & slots_mask] == -1) out[0] = acc;
}

template <typename F>
static int time_best(pct_ctx* ctx, F&& launch, double* best_ms) {
    cudaEvent_t e0, e1;
    PCT_CUDA(ctx, cudaEventCreate(&e0));
    PCT_CUDA(ctx, cudaEventCreate(&e1));
    *best_ms = 1e30;
    for (int rep = 0; rep < 4; ++rep) {
        PCT_CUDA(ctx, cudaEventRecord(e0, 0));
        launch();
        PCT_CUDA(ctx, cudaEventRecord(e1, 0));
        PCT_CUDA(ctx, cudaEventSynchronize(e1));
        PCT_CUDA(ctx, cudaGetLastError());
        float ms = 0.f;
        PCT_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < *best_ms) *best_ms = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return PCT_OK;
}

}  // namespace pct

using namespace pct;

extern "C" int pct_measure_peaks(pct_ctx* ctx, pct_peaks* out) {
    if (!ctx || !out) return PCT_E_INVALID_ARG;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(ctx->device);
    const int sms = ctx->num_sms;
    const unsigned n = 1u << 24;                      // 16 Mi floats = 64 MiB: L2-resident, like x of config 3
    float* buf = nullptr;
    int rc = PCT_OK;
    double ms = 0.0;
    auto done = [&](int code) { cudaFree(buf); if (prev >= 0) cudaSetDevice(prev); return code; };
    if (cudaMalloc(&buf, sizeof(float) * 2 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return done(set_error(ctx, PCT_E_OOM, "peaks buffer")); }
    cudaMemset(buf, 0, sizeof(float) * 2 * (size_t)n);
    {   // FP64 FMA
        const int blocks = sms * 8, iters = 4096;
        if ((rc = time_best(ctx, [&] { k_peak_fp64<<<blocks, PK_THREADS>>>((double*)buf, iters, 1.0000001, 1e-9); }, &ms)) != PCT_OK) return done(rc);
        out->fp64_fma_per_s = (double)blocks * PK_THREADS * iters * 8.0 / (ms * 1e-3);
    }
    {   // L2 gather
        const int blocks = sms * 16, iters = 256;
        if ((rc = time_best(ctx, [&] { k_peak_gather<<<blocks, PK_THREADS>>>(buf, n - 1, iters, buf); }, &ms)) != PCT_OK) return done(rc);
        out->l2_gather_per_s = (double)blocks * PK_THREADS * iters * 8.0 / (ms * 1e-3);
    }
    for (int mode = 0; mode < 3; ++mode) {            // L2 reductions
        const int blocks = sms * 16, iters = 1024;
        const unsigned mask = mode == 0 ? n - 1 : n - 1;   // mode >= 1 addresses float2 slots: n slots of 8 bytes (128 MiB)
        if ((rc = time_best(ctx, [&] { k_peak_red<<<blocks, PK_THREADS>>>(buf, mask, iters, mode); }, &ms)) != PCT_OK) return done(rc);
        const double rate = (double)blocks * PK_THREADS * iters / (ms * 1e-3);
        if (mode == 0) out->l2_red_f32_per_s = rate; else if (mode == 1) out->l2_red_v2_per_s = rate; else out->l2_red_v2_coalesced_per_s = rate;
    }
    for (int mode = 0; mode < 4; ++mode) {            // shared memory: 8192 slots, 1024 threads, 2 CTAs / SM
        const int blocks = sms * 2, iters = 2048, slots = 8192;
        if ((rc = time_best(ctx, [&] { k_peak_smem<<<blocks, 1024, slots * sizeof(int)>>>(slots - 1, iters, mode, (int*)buf); }, &ms)) != PCT_OK) return done(rc);
        const double rate = (double)blocks * 1024.0 * iters * 4.0 / (ms * 1e-3);
        if (mode == 0) out->smem_atomic_per_s = rate; else if (mode == 1) out->smem_load_per_s = rate;
        else if (mode == 2) out->smem_atomic_cf_per_s = rate; else out->smem_load_cf_per_s = rate;
    }
    out->num_sms = sms;
    return done(PCT_OK);
}
