// solve_kernels.cu -- K2/K3: projections along the encoded rows and the DROP block update (A4-A9).
// PAPER.md:98 (DROP, block = protons processed in parallel), PAPER.md:7 (b = A x); readings R12-R20.
//
// One warp per history.  Lane l of round r owns visit 32 r + l: every lane extracts its own 3-bit code from the
// row's 128-bit chunks (three 64-bit words cover 32 consecutive codes, so the loads are warp-broadcasts), turns it
// into a linear-index delta, and a warp inclusive scan yields all 32 voxel indices at once.  Consecutive lanes then
// touch consecutive voxels of the path, so gathers of x and reductions into {Delta,s} coalesce per 32-byte sector
// wherever the path runs along x.  The code stream is the only compulsory HBM traffic (3 bit / visit); x and the
// accumulator live in L2.
#include <cooperative_groups.h>

#include <climits>

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

// The same walk, four rounds (128 visits) at a time: all four rounds are decoded first, then `load` is issued for all of
// them, then `use` consumes the results -- the memory round trips of the four rounds overlap instead of following one
// another (a warp issues in order: it would stall at the first use of round r before issuing round r + 1).
template <typename T, typename L, typename U>
__device__ __forceinline__ void for_each_visit_x4(const ulonglong2* __restrict__ codes, uint64_t off, int32_t start, unsigned n,
                                                  int sx, int sy, int sz, int lane, L&& load, U&& use) {
    const unsigned long long* cp = reinterpret_cast<const unsigned long long*>(codes + off);
    int base = start;
    for (unsigned v0 = 0; v0 < n; v0 += 128) {
        int vox[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const unsigned visit = v0 + 32u * r + lane;
            int d = 0;
            if (visit < n && visit > 0) d = step_delta(cp, visit, sx, sy, sz);
            vox[r] = base + warp_inclusive_scan(d, lane);
            base = __shfl_sync(0xffffffffu, vox[r], 31);
        }
        T val[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) if (v0 + 32u * r + lane < n) val[r] = load(vox[r]);
#pragma unroll
        for (int r = 0; r < 4; ++r) if (v0 + 32u * r + lane < n) use(vox[r], val[r]);
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

// Bounding box {x0, y0, z0, x1, y1, z1} of the voxels a block visits (counts > 0), into box6 (pre-set to {large.., -1..}): the
// later sweeps over this block only look there (k_block_update_cached4_box).  One warp per grid row (y, z), lanes along x.
__global__ void __launch_bounds__(256) k_counts_bbox(const uint4* __restrict__ counts4, int nx4, int ny, int nz, int* __restrict__ box6) {
    const int lane = threadIdx.x & 31, rows = ny * nz;
    int lo0 = INT_MAX, hi0 = -1, lo1 = INT_MAX, hi1 = -1, lo2 = INT_MAX, hi2 = -1;
    for (int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); row < rows; row += gridDim.x * (blockDim.x >> 5)) {
        const uint4* c = counts4 + (size_t)row * nx4;
        int first = INT_MAX, last = -1;
        for (int q = lane; q < nx4; q += 32) {                 // 16 bytes per lane: 128 voxels of the row per warp and turn
            const uint4 v = __ldg(c + q);
            const unsigned m = (v.x ? 1u : 0u) | (v.y ? 2u : 0u) | (v.z ? 4u : 0u) | (v.w ? 8u : 0u);
            if (m) { first = min(first, 4 * q + __ffs(m) - 1); last = max(last, 4 * q + 31 - __clz(m)); }
        }
        first = __reduce_min_sync(0xffffffffu, first);
        last = __reduce_max_sync(0xffffffffu, last);
        if (last >= 0) {
            const int z = row / ny, y = row - z * ny;
            lo0 = min(lo0, first); hi0 = max(hi0, last); lo1 = min(lo1, y); hi1 = max(hi1, y); lo2 = min(lo2, z); hi2 = max(hi2, z);
        }
    }
    // one set of atomics per CTA (same-address atomics serialise in L2); the plain read filters out those that cannot change anything
    __shared__ int sh[6][8];
    if (lane == 0) { const int w = threadIdx.x >> 5; sh[0][w] = lo0; sh[1][w] = lo1; sh[2][w] = lo2; sh[3][w] = hi0; sh[4][w] = hi1; sh[5][w] = hi2; }
    __syncthreads();
    if (threadIdx.x < 6) {
        const int k = threadIdx.x;
        int v = sh[k][0];
        for (int w = 1; w < 8; ++w) v = k < 3 ? min(v, sh[k][w]) : max(v, sh[k][w]);
        volatile int* vb = box6;
        if (k < 3) { if (v < vb[k]) atomicMin(box6 + k, v); }
        else if (v > vb[k]) atomicMax(box6 + k, v);
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

// the same over the bounding box of the voxels the block visits (box6 of k_block_update_store; nx divisible by 4): a block's
// histories cover the object, not the grid -- on configs 2 / 3 a third of the voxels
__global__ void __launch_bounds__(256) k_block_update_cached4_box(float4* __restrict__ x, float4* __restrict__ dsum, int nx4, int ny, float lambda,
                                                                  const uint4* __restrict__ counts, Clamp cl, const int* __restrict__ box6) {
    const int x0 = __ldg(box6 + 0) >> 2, y0 = __ldg(box6 + 1), z0 = __ldg(box6 + 2);
    const int w = (__ldg(box6 + 3) >> 2) - x0 + 1, h = __ldg(box6 + 4) - y0 + 1, d = __ldg(box6 + 5) - z0 + 1;
    if (w <= 0 || h <= 0 || d <= 0) return;                  // the block visits nothing
    const int cells = w * h * d, stride = (int)(gridDim.x * blockDim.x);
    for (int q = (int)(blockIdx.x * blockDim.x + threadIdx.x); q < cells; q += stride) {
        const int r = q / w, xq = q - r * w, zz = r / h, yy = r - zz * h;
        const int64_t j = ((int64_t)(zz + z0) * ny + (yy + y0)) * nx4 + (x0 + xq);
        const float4 dl = dsum[j];
        const bool moved = !(dl.x == 0.f && dl.y == 0.f && dl.z == 0.f && dl.w == 0.f);
        if (!moved && !cl.on) continue;
        const uint4 c = counts[j];
        if (!moved && (c.x | c.y | c.z | c.w) == 0u) continue;
        float4 v = x[j];
        if (c.x > 0u) v.x = clamp_of(cl, dl.x != 0.f ? v.x + lambda * dl.x / (float)c.x : v.x);
        if (c.y > 0u) v.y = clamp_of(cl, dl.y != 0.f ? v.y + lambda * dl.y / (float)c.y : v.y);
        if (c.z > 0u) v.z = clamp_of(cl, dl.z != 0.f ? v.z + lambda * dl.z / (float)c.z : v.z);
        if (c.w > 0u) v.w = clamp_of(cl, dl.w != 0.f ? v.w + lambda * dl.w / (float)c.w : v.w);
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
// box6 (device, may be NULL): the block's visited bounding box, written by the storing sweep and used by the cached ones.
int launch_block_update(pct_ctx* ctx, float* x, float2* ds, float* dsum, uint32_t* counts, bool store, float lambda, float clamp_lo,
                        float clamp_hi, int* box6, cudaStream_t st) {
    const Clamp cl = {clamp_lo, clamp_hi, clamp_lo <= clamp_hi ? 1 : 0};
    const int64_t n = ctx->n_vox;
    const int64_t want = (n + 255) / 256;
    const int64_t cap = (int64_t)ctx->num_sms * 16;
    const unsigned grid = (unsigned)(want < cap ? want : cap);
    ProfScope prof(ctx, 2, st);
    if (!counts) k_block_update<<<grid, 256, 0, st>>>(x, ds, n, lambda, cl);
    else if (store) {
        k_block_update_store<<<grid, 256, 0, st>>>(x, ds, n, lambda, counts, cl);
        if (box6 && n < 0x7fffffffLL) {
            PCT_CUDA(ctx, cudaMemsetAsync(box6, 0x7f, 3 * sizeof(int), st));          // mins: a large int
            PCT_CUDA(ctx, cudaMemsetAsync(box6 + 3, 0xff, 3 * sizeof(int), st));      // maxes: -1
            if (ctx->geom.nx % 4 == 0 && ((uintptr_t)counts & 15) == 0) {         // the box kernel's own conditions
                const int rows = ctx->geom.ny * ctx->geom.nz;
                k_counts_bbox<<<(unsigned)min((rows + 7) / 8, ctx->num_sms * 4), 256, 0, st>>>(reinterpret_cast<const uint4*>(counts), ctx->geom.nx / 4, ctx->geom.ny,
                                                                         ctx->geom.nz, box6);
                ++ctx->launches;
            }
        }
    } else if (box6 && ctx->geom.nx % 4 == 0 && n < 0x7fffffffLL && (((uintptr_t)x | (uintptr_t)dsum | (uintptr_t)counts) & 15) == 0)
        k_block_update_cached4_box<<<grid, 256, 0, st>>>(reinterpret_cast<float4*>(x), reinterpret_cast<float4*>(dsum), ctx->geom.nx / 4, ctx->geom.ny,
                                                         lambda, reinterpret_cast<const uint4*>(counts), cl, box6);
    else if (n % 4 == 0 && (((uintptr_t)x | (uintptr_t)dsum | (uintptr_t)counts) & 15) == 0)
        k_block_update_cached4<<<grid, 256, 0, st>>>(reinterpret_cast<float4*>(x), reinterpret_cast<float4*>(dsum), n / 4, lambda,
                                                     reinterpret_cast<const uint4*>(counts), cl);
    else k_block_update_cached<<<grid, 256, 0, st>>>(x, dsum, n, lambda, counts, cl);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// ---- small blocks: all sweeps in ONE persistent cooperative kernel (A8; block 3200 is 2x slower than
// 320000) ------------------------------------------------------------------------------------------------------------------
// With a few thousand histories per block a sweep is tens of thousands of (project, update) pairs of a few microseconds
// each.  Launched pair by pair (from the host or from a CUDA graph: measured 19-21 us per pair either way at B = 1000) the
// sweep is bound by launch latency and by the chain of dependent loads every fresh kernel starts with, and an update pass
// over the whole grid per block adds n voxels x blocks of traffic.  Here the control never leaves the device:
//   * one cooperative kernel, as many CTAs as a block has work for (all co-resident), loops over iters x blocks; the two
//     phases of a block are separated by grid-wide barriers instead of kernel boundaries;
//   * the update does not sweep the grid: every warp walks its rows once more and, at every visit, claims the voxel's
//     accumulator with an atomic exchange -- the one visit that gets a non-zero count back applies
//     x_j += lambda Delta_j / s_j (and the clamp), all others see zero and pass.  The accumulator is left cleared;
//   * a warp keeps the same position in every block; the header of its first row of the next block is loaded, and the row's
//     codes are pulled into L2, before the barrier.
// x is read with ld.global.cg (L2): other SMs change it between the phases.
namespace cg = cooperative_groups;

struct RowHead { unsigned n; int32_t start; uint64_t off; float ell, b, w; };

__device__ __forceinline__ RowHead load_head(const uint32_t* __restrict__ N, const int32_t* __restrict__ start, const float* __restrict__ ell,
                                             const uint64_t* __restrict__ code_off, const float* __restrict__ b, const float* __restrict__ wts, int64_t i) {
    RowHead h;
    h.n = N[i]; h.start = start[i]; h.off = code_off[i]; h.ell = ell[i]; h.b = b[i]; h.w = wts ? wts[i] : 1.f;
    return h;
}

// 8 warps per CTA: 1024-thread CTAs (fewer arrivals at the grid barrier) were 35 % slower -- a block of 1000 rows then sits on 32 SMs
constexpr int PS_THREADS = 256, PS_WARPS = PS_THREADS / 32;

__global__ void __launch_bounds__(PS_THREADS)
k_sweeps_persistent(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const int32_t* __restrict__ start,
                    const float* __restrict__ ell, const uint64_t* __restrict__ code_off, const ulonglong2* __restrict__ codes, int64_t m,
                    int64_t block_size, int64_t n_blocks, int iters, const float* __restrict__ b, const float* __restrict__ wts, float* x,
                    float2* ds, float lambda, Clamp cl) {
    cg::grid_group grid = cg::this_grid();
    const int lane = threadIdx.x & 31;
    const int64_t warp = (int64_t)blockIdx.x * PS_WARPS + (threadIdx.x >> 5), warps = (int64_t)gridDim.x * PS_WARPS;
    const int64_t total = (int64_t)iters * n_blocks;
    // the header of the first row this warp takes in a block, loaded one block ahead (and its codes pulled into L2)
    auto first_row = [&](int64_t pair) { const int64_t t = pair % n_blocks; return t * block_size + warp; };
    auto row_end = [&](int64_t pair) { const int64_t i0 = (pair % n_blocks) * block_size; return (m - i0) < block_size ? m : i0 + block_size; };
    RowHead next = {};
    if (first_row(0) < row_end(0)) next = load_head(N, start, ell, code_off, b, wts, first_row(0));
    for (int64_t pair = 0; pair < total; ++pair) {
        const int64_t i1 = row_end(pair);
        // A5 + A6: project and scatter
        for (int64_t i = first_row(pair); i < i1; i += warps) {
            const RowHead h = i == first_row(pair) ? next : load_head(N, start, ell, code_off, b, wts, i);
            if (h.n == 0) continue;
            float S = 0.f;
            for_each_visit_x4<float>(codes, h.off, h.start, h.n, g.sx, g.sy, g.sz, lane, [&](int vox) { return __ldcg(x + vox); },
                                     [&](int, float v) { S += v; });
            S = warp_sum(S);
            const float c = h.w * (h.b - h.ell * S) / ((float)h.n * h.ell);
            for_each_visit(codes, h.off, h.start, h.n, g.sx, g.sy, g.sz, lane, [&](int vox) { red_add_v2(ds + vox, c, 1.0f); });
        }
        grid.sync();
        // A7: the visit that still finds the count owns the voxel's update.  One 64-bit exchange fetches and clears
        // {Delta_j, s_j}; x_j is loaded alongside it rather than after it.
        for (int64_t i = first_row(pair); i < i1; i += warps) {
            const RowHead h = i == first_row(pair) ? next : load_head(N, start, ell, code_off, b, wts, i);
            if (h.n == 0) continue;
            struct Got { float xv; unsigned long long old; };
            for_each_visit_x4<Got>(codes, h.off, h.start, h.n, g.sx, g.sy, g.sz, lane,
                                   [&](int vox) { Got q; q.xv = __ldcg(x + vox); q.old = atomicExch(reinterpret_cast<unsigned long long*>(ds + vox), 0ull); return q; },
                                   [&](int vox, const Got& q) {
                                       const float s = __uint_as_float((unsigned)(q.old >> 32)), d = __uint_as_float((unsigned)q.old);
                                       if (s > 0.f) x[vox] = clamp_of(cl, q.xv + lambda * d / s);
                                   });
        }
        if (pair + 1 < total && first_row(pair + 1) < row_end(pair + 1)) {
            next = load_head(N, start, ell, code_off, b, wts, first_row(pair + 1));
            const char* cp = reinterpret_cast<const char*>(codes + next.off);
            if (next.n > 0 && (unsigned)lane * 128u < (next.n * 3u + 7u) / 8u) asm volatile("prefetch.global.L2 [%0];" ::"l"(cp + lane * 128));
        }
        grid.sync();
    }
}

// iters sweeps over all blocks of `block_size` histories in one cooperative launch.  ds must be all zero (it is left so).
// Returns PCT_E_CAPACITY (and sets no error text) if the device cannot launch cooperatively: the caller falls back.
int launch_sweeps_persistent(pct_ctx* ctx, const pct_paths* P, const float* b, const float* wts, float* x, int iters, int64_t block_size, float lambda,
                             float clamp_lo, float clamp_hi, cudaStream_t st) {
    int64_t n_blocks = (P->m + block_size - 1) / block_size;
    if (iters <= 0 || n_blocks == 0) return PCT_OK;
    int coop = 0, per_sm = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
    if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sweeps_persistent, PS_THREADS, 0) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return PCT_E_CAPACITY;
    }
    Clamp cl = {clamp_lo, clamp_hi, clamp_lo <= clamp_hi ? 1 : 0};
    const int64_t rows = block_size < P->m ? block_size : P->m;
    const int64_t want = (rows + PS_WARPS - 1) / PS_WARPS, cap = (int64_t)ctx->num_sms * per_sm;
    int grid = (int)(want < cap ? want : cap);
    if (grid < 1) grid = 1;
    int64_t m = P->m;
    const uint32_t* N = P->N; const int32_t* start = P->start; const float* ell = P->ell; const uint64_t* code_off = P->code_off;
    const ulonglong2* codes = P->codes; float2* ds = ctx->ds;
    void* args[] = {(void*)&ctx->cfg, (void*)&N, (void*)&start, (void*)&ell, (void*)&code_off, (void*)&codes, (void*)&m, (void*)&block_size,
                    (void*)&n_blocks, (void*)&iters, (void*)&b, (void*)&wts, (void*)&x, (void*)&ds, (void*)&lambda, (void*)&cl};
    ProfScope prof(ctx, 3, st);
    PCT_CUDA(ctx, cudaLaunchCooperativeKernel((const void*)k_sweeps_persistent, dim3((unsigned)grid), dim3(PS_THREADS), args, 0, st));
    ++ctx->launches;
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
