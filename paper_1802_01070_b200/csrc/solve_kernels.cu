// solve_kernels.cu -- K2/K3: projections along the encoded rows and the DROP block update (A4-A9).
// PAPER.md:98 (DROP, block = protons processed in parallel), PAPER.md:7 (b = A x); readings R12-R20.
//
// One warp per history.  Lane l of round r owns visit 32 r + l: every lane extracts its own 3-bit code from the
// row's 128-bit chunks (three 64-bit words cover 32 consecutive codes, so the loads are warp-broadcasts), turns it
// into a linear-index delta, and a warp inclusive scan yields all 32 voxel indices at once.  Consecutive lanes then
// touch consecutive voxels of the path, so gathers of x and reductions into {Delta,s} coalesce per 32-byte sector
// wherever the path runs along x.  The code stream is the only compulsory HBM traffic (3 bit / visit); x and the
// accumulator live in L2.
#include "pct_internal.cuh"

namespace pct {

constexpr int PROJ_THREADS = 256;
constexpr int PROJ_WARPS = PROJ_THREADS / 32;

__device__ __forceinline__ int warp_inclusive_scan(int v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += y;
    }
    return v;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// linear-index delta of the step INTO visit `visit` (visit >= 1) of a row whose codes start at cp
__device__ __forceinline__ int step_delta(const unsigned long long* __restrict__ cp, unsigned visit, int sx, int sy, int sz) {
    const unsigned ci = visit - 1u;
    const unsigned word = ci / CODES_PER_WORD, sh = 3u * (ci % CODES_PER_WORD);
    const int code = (int)((__ldg(cp + word) >> sh) & 7ull);
    const int axis = code >> 1;
    const int mag = axis == 0 ? sx : (axis == 1 ? sy : sz);
    return (code & 1) ? -mag : mag;
}

// Walks the row of history i; calls f(voxel) on every lane that owns a visit.  All 32 lanes must call.
template <typename F>
__device__ __forceinline__ void for_each_visit(const ulonglong2* __restrict__ codes, uint64_t off, int32_t start, unsigned n,
                                               int sx, int sy, int sz, int lane, F&& f) {
    const unsigned long long* cp = reinterpret_cast<const unsigned long long*>(codes + off);
    int base = start;
    for (unsigned v0 = 0; v0 < n; v0 += 32) {
        const unsigned visit = v0 + lane;
        int d = 0;
        if (visit < n && visit > 0) d = step_delta(cp, visit, sx, sy, sz);
        const int vox = base + warp_inclusive_scan(d, lane);
        if (visit < n) f(vox);
        base = __shfl_sync(0xffffffffu, vox, 31);
    }
}

// A9 / R19
__global__ void __launch_bounds__(PROJ_THREADS)
k_forward_project(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const int32_t* __restrict__ start,
                  const float* __restrict__ ell, const uint64_t* __restrict__ code_off, const ulonglong2* __restrict__ codes,
                  int64_t m, const float* __restrict__ x, float* __restrict__ b_out) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = (int64_t)gridDim.x * PROJ_WARPS;
    for (int64_t i = (int64_t)blockIdx.x * PROJ_WARPS + (threadIdx.x >> 5); i < m; i += warps) {
        const unsigned n = N[i];
        float S = 0.f;
        if (n > 0)
            for_each_visit(codes, code_off[i], start[i], n, g.sx, g.sy, g.sz, lane, [&](int vox) { S += __ldg(x + vox); });
        S = warp_sum(S);
        if (lane == 0) b_out[i] = n > 0 ? ell[i] * S : 0.f;
    }
}

// A4 / R20
__global__ void __launch_bounds__(PROJ_THREADS)
k_column_counts(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const int32_t* __restrict__ start,
                const uint64_t* __restrict__ code_off, const ulonglong2* __restrict__ codes, int64_t i0, int64_t i1,
                uint32_t* __restrict__ counts) {
    const int lane = threadIdx.x & 31;
    const int64_t warps = (int64_t)gridDim.x * PROJ_WARPS;
    for (int64_t i = i0 + (int64_t)blockIdx.x * PROJ_WARPS + (threadIdx.x >> 5); i < i1; i += warps) {
        const unsigned n = N[i];
        if (n > 0)
            for_each_visit(codes, code_off[i], start[i], n, g.sx, g.sy, g.sz, lane, [&](int vox) { atomicAdd(counts + vox, 1u); });
    }
}

__device__ __forceinline__ void red_add_v2(float2* p, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

// A5 + A6 (+A4 fused): for every history of the block, S_i = sum x_j (gather), c_i = (b_i - l_i S_i)/(N_i l_i) (R17),
// then {Delta_j, s_j} += {c_i, 1} on every visit.  x is frozen during the block (R14): it is only read here.
// COUNT = false: the block's column counts are cached (R15: they do not depend on x); only Delta_j is accumulated.
template <bool COUNT>
__global__ void __launch_bounds__(PROJ_THREADS)
k_block_project_scatter(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const int32_t* __restrict__ start,
                        const float* __restrict__ ell, const uint64_t* __restrict__ code_off,
                        const ulonglong2* __restrict__ codes, int64_t i0, int64_t i1, const uint32_t* __restrict__ list,
                        const float* __restrict__ b, const float* __restrict__ wts, const float* __restrict__ x, float2* __restrict__ ds,
                        float* __restrict__ dsum) {
    // list == nullptr: histories [i0, i1); else the histories list[i0 .. i1) (a block's direct list, plan.cu)
    const int lane = threadIdx.x & 31;
    const int64_t warps = (int64_t)gridDim.x * PROJ_WARPS;
    for (int64_t k = i0 + (int64_t)blockIdx.x * PROJ_WARPS + (threadIdx.x >> 5); k < i1; k += warps) {
        const int64_t i = list ? (int64_t)list[k] : k;
        const unsigned n = N[i];
        if (n == 0) continue;
        const uint64_t off = code_off[i];
        const int32_t st = start[i];
        float S = 0.f;
        for_each_visit(codes, off, st, n, g.sx, g.sy, g.sz, lane, [&](int vox) { S += __ldg(x + vox); });
        S = warp_sum(S);
        const float l = ell[i];
        float c = (b[i] - l * S) / ((float)n * l);
        if (wts) c *= wts[i];                                   // R27: weighted row
        for_each_visit(codes, off, st, n, g.sx, g.sy, g.sz, lane, [&](int vox) {
            if (COUNT) red_add_v2(ds + vox, c, 1.0f);
            else asm volatile("red.global.add.f32 [%0], %1;" ::"l"(dsum + vox), "f"(c) : "memory");
        });
    }
}

// A7: x_j += lambda * Delta_j / max(1, s_j); clear the accumulator (R15-R16).  Only touched voxels are written.
// clamp_of: R27's box clamp on an updated voxel (NaN stays NaN: it is compared, not passed through fminf / fmaxf)
struct Clamp { float lo, hi; int on; };
__device__ __forceinline__ float clamp_of(const Clamp& c, float v) { return c.on ? (v < c.lo ? c.lo : (v > c.hi ? c.hi : v)) : v; }

__global__ void __launch_bounds__(256) k_block_update(float* __restrict__ x, float2* __restrict__ ds, int64_t n, float lambda, Clamp cl) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        const float2 a = ds[j];
        if (a.y > 0.f) {
            x[j] = clamp_of(cl, x[j] + lambda * a.x / a.y);
            ds[j] = make_float2(0.f, 0.f);
        }
    }
}

// A7, first sweep over a block with a count cache: as k_block_update, and s_j^t is stored (all voxels: zeros too).
__global__ void __launch_bounds__(256) k_block_update_store(float* __restrict__ x, float2* __restrict__ ds, int64_t n, float lambda,
                                                            uint32_t* __restrict__ counts, Clamp cl) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        const float2 a = ds[j];
        counts[j] = (uint32_t)a.y;
        if (a.y > 0.f) {
            x[j] = clamp_of(cl, x[j] + lambda * a.x / a.y);
            ds[j] = make_float2(0.f, 0.f);
        }
    }
}

// A7 with cached counts: x_j += lambda * Delta_j / s_j^t wherever Delta_j != 0 (a zero sum leaves x_j unchanged anyway).
// With the clamp on, every voxel the block visits (s_j^t > 0) is clamped, moved or not (R27), so the counts are read for all.
__global__ void __launch_bounds__(256) k_block_update_cached(float* __restrict__ x, float* __restrict__ dsum, int64_t n, float lambda,
                                                             const uint32_t* __restrict__ counts, Clamp cl) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        const float d = dsum[j];
        if (d != 0.f) {
            x[j] = clamp_of(cl, x[j] + lambda * d / (float)counts[j]);
            dsum[j] = 0.f;
        } else if (cl.on && counts[j] > 0u) {
            x[j] = clamp_of(cl, x[j]);
        }
    }
}

// the same, four voxels per thread with 16-byte accesses (n divisible by 4, pointers 16-byte aligned)
__global__ void __launch_bounds__(256) k_block_update_cached4(float4* __restrict__ x, float4* __restrict__ dsum, int64_t n4, float lambda,
                                                              const uint4* __restrict__ counts, Clamp cl) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n4; j += stride) {
        const float4 d = dsum[j];
        const bool moved = !(d.x == 0.f && d.y == 0.f && d.z == 0.f && d.w == 0.f);
        if (!moved && !cl.on) continue;
        const uint4 c = counts[j];
        if (!moved && (c.x | c.y | c.z | c.w) == 0u) continue;
        float4 v = x[j];
        if (c.x > 0u) v.x = clamp_of(cl, d.x != 0.f ? v.x + lambda * d.x / (float)c.x : v.x);
        if (c.y > 0u) v.y = clamp_of(cl, d.y != 0.f ? v.y + lambda * d.y / (float)c.y : v.y);
        if (c.z > 0u) v.z = clamp_of(cl, d.z != 0.f ? v.z + lambda * d.z / (float)c.z : v.z);
        if (c.w > 0u) v.w = clamp_of(cl, d.w != 0.f ? v.w + lambda * d.w / (float)c.w : v.w);
        x[j] = v;
        if (moved) dsum[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

__global__ void __launch_bounds__(256) k_fill(float* __restrict__ p, int64_t n, float value) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) p[j] = value;
}

static int proj_grid(const pct_ctx* ctx, int64_t rows) {
    const int64_t want = (rows + PROJ_WARPS - 1) / PROJ_WARPS;
    const int64_t cap = (int64_t)ctx->num_sms * 8;      // 8 resident CTAs of 256 threads per SM, grid-stride beyond
    return (int)(want < 1 ? 1 : (want < cap ? want : cap));
}

int launch_forward_project(pct_ctx* ctx, const pct_paths* P, const float* x, float* b_out, cudaStream_t st) {
    if (P->m <= 0) return PCT_OK;
    k_forward_project<<<proj_grid(ctx, P->m), PROJ_THREADS, 0, st>>>(ctx->cfg, P->N, P->start, P->ell, P->code_off,
                                                                     P->codes, P->m, x, b_out);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

int launch_column_counts(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, uint32_t* counts, cudaStream_t st) {
    PCT_CUDA(ctx, cudaMemsetAsync(counts, 0, sizeof(uint32_t) * (size_t)P->n_vox, st));
    if (i1 <= i0) return PCT_OK;
    k_column_counts<<<proj_grid(ctx, i1 - i0), PROJ_THREADS, 0, st>>>(ctx->cfg, P->N, P->start, P->code_off, P->codes, i0,
                                                                      i1, counts);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

int launch_block_project_scatter(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, const uint32_t* list, bool count,
                                 const float* b, const float* wts, const float* x, float2* ds, float* dsum, cudaStream_t st) {
    if (i1 <= i0) return PCT_OK;
    ProfScope prof(ctx, 3, st);
    if (count)
        k_block_project_scatter<true><<<proj_grid(ctx, i1 - i0), PROJ_THREADS, 0, st>>>(ctx->cfg, P->N, P->start, P->ell, P->code_off,
                                                                                        P->codes, i0, i1, list, b, wts, x, ds, dsum);
    else
        k_block_project_scatter<false><<<proj_grid(ctx, i1 - i0), PROJ_THREADS, 0, st>>>(ctx->cfg, P->N, P->start, P->ell, P->code_off,
                                                                                         P->codes, i0, i1, list, b, wts, x, ds, dsum);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// counts == nullptr: fused counts in ds.  store: fused counts, and s_j is written to counts.  else: cached counts, dsum.
int launch_block_update(pct_ctx* ctx, float* x, float2* ds, float* dsum, uint32_t* counts, bool store, float lambda, float clamp_lo,
                        float clamp_hi, cudaStream_t st) {
    const Clamp cl = {clamp_lo, clamp_hi, clamp_lo <= clamp_hi ? 1 : 0};
    const int64_t n = ctx->n_vox;
    const int64_t want = (n + 255) / 256;
    const int64_t cap = (int64_t)ctx->num_sms * 16;
    const unsigned grid = (unsigned)(want < cap ? want : cap);
    ProfScope prof(ctx, 2, st);
    if (!counts) k_block_update<<<grid, 256, 0, st>>>(x, ds, n, lambda, cl);
    else if (store) k_block_update_store<<<grid, 256, 0, st>>>(x, ds, n, lambda, counts, cl);
    else if (n % 4 == 0 && (((uintptr_t)x | (uintptr_t)dsum | (uintptr_t)counts) & 15) == 0)
        k_block_update_cached4<<<grid, 256, 0, st>>>(reinterpret_cast<float4*>(x), reinterpret_cast<float4*>(dsum), n / 4, lambda,
                                                     reinterpret_cast<const uint4*>(counts), cl);
    else k_block_update_cached<<<grid, 256, 0, st>>>(x, dsum, n, lambda, counts, cl);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

int launch_fill(pct_ctx* ctx, float* p, int64_t n, float value, cudaStream_t st) {
    if (n <= 0) return PCT_OK;
    const int64_t want = (n + 255) / 256, cap = (int64_t)ctx->num_sms * 16;
    k_fill<<<(unsigned)(want < cap ? want : cap), 256, 0, st>>>(p, n, value);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

}  // namespace pct
