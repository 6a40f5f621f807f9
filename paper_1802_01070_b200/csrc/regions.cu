// regions.cu -- Algorithm 1 of the paper, "multi-GPU based reconstruction" (reading R28 of DESIGN.md):
//   1: setupImageRegions()  2: identifyProtonsPassingRegions()  3: allocateMemoryForProtonsPerGPU()
//   4: iterativelySolvePerGPU()  5: selectSlice()
// The volume is cut along z into overlapping regions, every region is solved on the histories that enter or leave it, with no
// exchange between the regions; the final image takes every slice from the region whose own (non-overlapped) part holds it.
// Step 4 is the single-GPU path of this library unchanged (pct_generate_mlp + pct_solve on the region's histories); the steps
// around it are the small kernels below.
#include <cub/cub.cuh>
#include <thrust/iterator/counting_iterator.h>

#include "pct_internal.cuh"

namespace pct {

// step 2: flag = 1 if the history was accepted by A1 and its entry slice or its exit slice lies in [z_lo, z_hi)
__global__ void __launch_bounds__(256)
k_region_flags(const int32_t* __restrict__ v_in, const int32_t* __restrict__ v_out, int64_t m, int slice, int z_lo, int z_hi,
               uint8_t* __restrict__ flag) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const int a = v_in[i], b = v_out[i];
    bool in = false;
    if (a >= 0 && b >= 0) {
        const int za = a / slice, zb = b / slice;
        in = (za >= z_lo && za < z_hi) || (zb >= z_lo && zb < z_hi);
    }
    flag[i] = in ? 1 : 0;
}

// step 3: nine tracker arrays and b, gathered
__global__ void __launch_bounds__(256)
k_gather_histories(const ProtonPtrs src, const float* __restrict__ b_src, const uint32_t* __restrict__ idx, int64_t count,
                   double* __restrict__ d0, double* __restrict__ d1, double* __restrict__ d2, double* __restrict__ d3,
                   double* __restrict__ d4, double* __restrict__ d5, double* __restrict__ d6, double* __restrict__ d7,
                   double* __restrict__ d8, float* __restrict__ b_dst) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    const uint32_t i = idx[k];
    d0[k] = src.phi[i]; d1[k] = src.t_in[i]; d2[k] = src.v_in[i]; d3[k] = src.dt_in[i]; d4[k] = src.dv_in[i];
    d5[k] = src.t_out[i]; d6[k] = src.v_out[i]; d7[k] = src.dt_out[i]; d8[k] = src.dv_out[i];
    if (b_dst) b_dst[k] = b_src[i];
}

}  // namespace pct

using namespace pct;

extern "C" {

int pct_regions_setup(int32_t nz, int32_t n_regions, int32_t ext, pct_region* out) {
    if (!out || nz < 1 || n_regions < 1 || n_regions > nz || ext < 0) return PCT_E_INVALID_ARG;
    for (int g = 0; g < n_regions; ++g) {
        const int lo = (int)((int64_t)g * nz / n_regions), hi = (int)((int64_t)(g + 1) * nz / n_regions);
        out[g].keep_lo = lo; out[g].keep_hi = hi;
        out[g].z_lo = g == 0 ? 0 : (lo - ext > 0 ? lo - ext : 0);
        out[g].z_hi = g == n_regions - 1 ? nz : (hi + ext < nz ? hi + ext : nz);
    }
    return PCT_OK;
}

int pct_hull_intersect(pct_ctx* ctx, const pct_protons* pr, const uint8_t* hull, int32_t* v_in, int32_t* v_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    int rc;
    if ((rc = check_protons(ctx, pr)) != PCT_OK) return rc;
    if (pr->m > 0 && (!v_in || !v_out)) return set_error(ctx, PCT_E_INVALID_ARG, "NULL output");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = prepare_hull_search(ctx, pr, hull, st)) != PCT_OK) return rc;
    const ProtonPtrs pp = {pr->phi, pr->t_in, pr->v_in, pr->dt_in, pr->dv_in, pr->t_out, pr->v_out, pr->dt_out, pr->dv_out};
    for (int64_t i0 = 0; i0 < pr->m; i0 += GEN_BATCH) {
        const int count = (int)((pr->m - i0) < GEN_BATCH ? (pr->m - i0) : GEN_BATCH);
        if ((rc = launch_hull_batch(ctx, pp, hull, i0, count, v_in, v_out, st)) != PCT_OK) return rc;
    }
    PCT_CUDA(ctx, cudaStreamSynchronize(st));
    return PCT_OK;
}

int pct_region_members(pct_ctx* ctx, const int32_t* v_in, const int32_t* v_out, int64_t m, const pct_region* region,
                       uint32_t* idx_out, int64_t* count_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!region || !count_out || m < 0 || m >= 0x7fffffffLL || (m > 0 && (!v_in || !v_out || !idx_out)))
        return set_error(ctx, PCT_E_INVALID_ARG, "bad region_members arguments");
    *count_out = 0;
    if (m == 0) return PCT_OK;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t* flag = nullptr;
    void* tmp = nullptr;
    int* d_count = nullptr;
    auto done = [&](int code) { cudaStreamSynchronize(st); cache_free(flag); cache_free(tmp); cache_free(d_count); return code; };
#define REG_CUDA(call)                                                                                          \
    do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError();                               \
        return done(set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
    REG_CUDA(cache_alloc((void**)&flag, (size_t)m));
    REG_CUDA(cache_alloc((void**)&d_count, 16));
    k_region_flags<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(v_in, v_out, m, ctx->geom.nx * ctx->geom.ny, region->z_lo, region->z_hi, flag);
    // stable compaction of the indices 0..m-1 by the flags: a library primitive, like the sorts
    thrust::counting_iterator<uint32_t> ids(0u);
    size_t tmp_bytes = 0;
    REG_CUDA(cub::DeviceSelect::Flagged(nullptr, tmp_bytes, ids, flag, idx_out, d_count, (int)m, st));
    REG_CUDA(cache_alloc(&tmp, tmp_bytes > 0 ? tmp_bytes : 16));
    REG_CUDA(cub::DeviceSelect::Flagged(tmp, tmp_bytes, ids, flag, idx_out, d_count, (int)m, st));
    int h_count = 0;
    REG_CUDA(cudaMemcpyAsync(&h_count, d_count, sizeof(int), cudaMemcpyDeviceToHost, st));
    REG_CUDA(cudaStreamSynchronize(st));
    REG_CUDA(cudaGetLastError());
#undef REG_CUDA
    ctx->launches += 3;
    *count_out = h_count;
    return done(PCT_OK);
}

int pct_gather_histories(pct_ctx* ctx, const pct_protons* src, const float* b_src, const uint32_t* idx, int64_t count,
                         pct_protons* dst, float* b_dst, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    int rc;
    if ((rc = check_protons(ctx, src)) != PCT_OK) return rc;
    if (!dst || count < 0 || count > src->m || (count > 0 && !idx) || ((b_src == nullptr) != (b_dst == nullptr)))
        return set_error(ctx, PCT_E_INVALID_ARG, "bad gather arguments");
    double* d[9] = {const_cast<double*>(dst->phi), const_cast<double*>(dst->t_in), const_cast<double*>(dst->v_in),
                    const_cast<double*>(dst->dt_in), const_cast<double*>(dst->dv_in), const_cast<double*>(dst->t_out),
                    const_cast<double*>(dst->v_out), const_cast<double*>(dst->dt_out), const_cast<double*>(dst->dv_out)};
    if (count > 0)
        for (int k = 0; k < 9; ++k)
            if (!d[k]) return set_error(ctx, PCT_E_INVALID_ARG, "NULL destination array");
    dst->m = count; dst->u_in_mm = src->u_in_mm; dst->u_out_mm = src->u_out_mm;
    if (count == 0) return PCT_OK;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const ProtonPtrs pp = {src->phi, src->t_in, src->v_in, src->dt_in, src->dv_in, src->t_out, src->v_out, src->dt_out, src->dv_out};
    k_gather_histories<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(pp, b_src, idx, count, d[0], d[1], d[2], d[3], d[4], d[5], d[6], d[7], d[8], b_dst);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

int pct_select_slices(pct_ctx* ctx, const float* x_region, const pct_region* region, float* x_final, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!x_region || !region || !x_final || region->keep_lo < 0 || region->keep_hi > ctx->geom.nz || region->keep_lo > region->keep_hi)
        return set_error(ctx, PCT_E_INVALID_ARG, "bad select_slices arguments");
    DeviceGuard guard(ctx->device);
    const size_t slice = (size_t)ctx->geom.nx * ctx->geom.ny;
    const size_t off = slice * (size_t)region->keep_lo, cnt = slice * (size_t)(region->keep_hi - region->keep_lo);
    if (cnt > 0 && x_region != x_final)
        PCT_CUDA(ctx, cudaMemcpyAsync(x_final + off, x_region + off, cnt * sizeof(float), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return PCT_OK;
}

int pct_reconstruct_regions(pct_ctx* ctx, const pct_protons* pr, const float* b, const uint8_t* hull, const float* x0,
                            int32_t n_regions, int32_t ext, int32_t region_first, int32_t region_count, int iters,
                            int64_t block_size, float lambda, float* x_out, int64_t* members_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    int rc;
    if ((rc = check_protons(ctx, pr)) != PCT_OK) return rc;
    if (!x_out || x_out == x0 || (pr->m > 0 && !b) || n_regions < 1 || n_regions > ctx->geom.nz || n_regions > 1024 || ext < 0 ||
        region_first < 0 || region_count < 0 || region_first + region_count > n_regions)
        return set_error(ctx, PCT_E_INVALID_ARG, "bad reconstruct_regions arguments");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    pct_region regions[1024];
    if (pct_regions_setup(ctx->geom.nz, n_regions, ext, regions) != PCT_OK) return set_error(ctx, PCT_E_INVALID_ARG, "bad regions");
    const int64_t m = pr->m;
    const size_t mm = (size_t)(m > 0 ? m : 1);
    int32_t *v_in = nullptr, *v_out = nullptr;
    uint32_t* idx = nullptr;
    double* arr[9] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    float *b_g = nullptr, *x_g = nullptr;
    pct_paths* P = nullptr;
    auto done = [&](int code) {
        cudaStreamSynchronize(st);
        if (P) pct_paths_free(P);
        cache_free(v_in); cache_free(v_out); cache_free(idx); cache_free(b_g); cache_free(x_g);
        for (int k = 0; k < 9; ++k) cache_free(arr[k]);
        return code;
    };
#define REG_CUDA(call)                                                                                          \
    do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError();                               \
        return done(set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
    REG_CUDA(cache_alloc((void**)&v_in, 4 * mm));
    REG_CUDA(cache_alloc((void**)&v_out, 4 * mm));
    REG_CUDA(cache_alloc((void**)&idx, 4 * mm));
    REG_CUDA(cache_alloc((void**)&x_g, sizeof(float) * (size_t)ctx->n_vox));
    if ((rc = pct_hull_intersect(ctx, pr, hull, v_in, v_out, stream)) != PCT_OK) return done(rc);        // A1 on all histories
    for (int g = region_first; g < region_first + region_count; ++g) {
        int64_t count = 0;
        if ((rc = pct_region_members(ctx, v_in, v_out, m, &regions[g], idx, &count, stream)) != PCT_OK) return done(rc);   // step 2
        if (members_out) members_out[g] = count;
        // step 3: the region's own copy of its histories (sized for this region; the cache reuses blocks of equal size)
        const size_t cc = (size_t)(count > 0 ? count : 1);
        for (int k = 0; k < 9; ++k) { cache_free(arr[k]); arr[k] = nullptr; }
        cache_free(b_g); b_g = nullptr;
        for (int k = 0; k < 9; ++k) REG_CUDA(cache_alloc((void**)&arr[k], sizeof(double) * cc));
        REG_CUDA(cache_alloc((void**)&b_g, sizeof(float) * cc));
        pct_protons sub = {count, arr[0], arr[1], arr[2], arr[3], arr[4], arr[5], arr[6], arr[7], arr[8], pr->u_in_mm, pr->u_out_mm};
        if ((rc = pct_gather_histories(ctx, pr, b, idx, count, &sub, b_g, stream)) != PCT_OK) return done(rc);
        // step 4: the single-GPU path on the region's histories
        if ((rc = pct_generate_mlp(ctx, &sub, hull, stream, &P)) != PCT_OK) return done(rc);
        if (!x0 && (rc = launch_fill(ctx, x_g, ctx->n_vox, 1.0f, st)) != PCT_OK) return done(rc);                 // x0 = 1
        if ((rc = pct_solve(ctx, P, b_g, x0 ? x0 : x_g, iters, block_size, lambda, x_g, stream)) != PCT_OK) return done(rc);
        if ((rc = pct_select_slices(ctx, x_g, &regions[g], x_out, stream)) != PCT_OK) return done(rc);          // step 5
        REG_CUDA(cudaStreamSynchronize(st));
        pct_paths_free(P); P = nullptr;
    }
#undef REG_CUDA
    return done(PCT_OK);
}

}  // extern "C"
