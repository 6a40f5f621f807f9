// pct_api.cu -- the extern "C" boundary of libpct.so (include/pct.h) and the iteration driver (A8).
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <unordered_map>

#include "pct_internal.cuh"

namespace pct {

// ---- size-keyed cache of device buffers --------------------------------------------------------------------------------
// Paths, plans and their scratch are rebuilt for every reconstruction with exactly the same sizes.  cudaMalloc/cudaFree of
// tens of GB costs hundreds of milliseconds, and the stream-ordered pool (cudaMallocAsync) reused such blocks erratically
// (35-700 ms per allocation, profiles/r01e_final.md).  So: freed blocks are kept per device and handed out again on an
// exact size match.  The cache is process-wide (buffers outlive contexts), trimmed when it exceeds half of the device
// memory or when an allocation fails, and by cache_trim().  A reused block is only safe because all work of a
// reconstruction is enqueued on one stream, in order.
namespace {
struct DevCache {
    std::mutex mu;
    std::unordered_map<void*, size_t> live;                    // blocks handed out
    std::unordered_multimap<size_t, void*> idle;               // blocks waiting for reuse
    size_t idle_bytes = 0;
};
DevCache& dev_cache(int device) {
    static DevCache caches[64];
    return caches[device >= 0 && device < 64 ? device : 0];
}
void trim_locked(DevCache& c) {
    for (auto& kv : c.idle) cudaFree(kv.second);
    c.idle.clear();
    c.idle_bytes = 0;
}
}  // namespace

cudaError_t cache_alloc(void** p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) bytes = 16;
    int device = 0;
    cudaGetDevice(&device);
    DevCache& c = dev_cache(device);
    std::lock_guard<std::mutex> lock(c.mu);
    auto it = c.idle.find(bytes);
    if (it != c.idle.end()) {
        *p = it->second;
        c.idle.erase(it);
        c.idle_bytes -= bytes;
        c.live[*p] = bytes;
        return cudaSuccess;
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {                 // make room and try once more
        cudaGetLastError();
        cudaDeviceSynchronize();
        trim_locked(c);
        e = cudaMalloc(p, bytes);
    }
    if (e == cudaSuccess) c.live[*p] = bytes;
    return e;
}

cudaError_t cache_free(void* p) {
    if (!p) return cudaSuccess;
    int device = 0;
    cudaGetDevice(&device);
    DevCache& c = dev_cache(device);
    std::lock_guard<std::mutex> lock(c.mu);
    auto it = c.live.find(p);
    if (it == c.live.end()) return cudaFree(p);          // not ours
    const size_t bytes = it->second;
    c.live.erase(it);
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && c.idle_bytes + bytes > total_b / 2) {
        cudaDeviceSynchronize();
        trim_locked(c);
    }
    c.idle.emplace(bytes, p);
    c.idle_bytes += bytes;
    return cudaSuccess;
}

void cache_trim(int device) {
    DevCache& c = dev_cache(device);
    std::lock_guard<std::mutex> lock(c.mu);
    cudaDeviceSynchronize();
    trim_locked(c);
}

int set_error(pct_ctx* ctx, int code, const char* fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

// events come from a per-context pool (creating one per launch would cost more than the short kernels it brackets)
static bool pool_get(pct_ctx* ctx, cudaEvent_t* e) {
    if (!ctx->prof_pool->empty()) { *e = ctx->prof_pool->back(); ctx->prof_pool->pop_back(); return true; }
    return cudaEventCreate(e) == cudaSuccess;
}
ProfScope::ProfScope(pct_ctx* c, int k, cudaStream_t s) : ctx(c), kind(k), st(s), on(c && c->profiling) {
    if (!on) return;
    cudaEvent_t e;
    if (!pool_get(ctx, &e)) { on = false; return; }
    cudaEventRecord(e, st);
    ctx->prof_events[kind]->push_back(e);
}
ProfScope::~ProfScope() {
    if (!on) return;
    cudaEvent_t e;
    if (!pool_get(ctx, &e)) { ctx->prof_pool->push_back(ctx->prof_events[kind]->back()); ctx->prof_events[kind]->pop_back(); return; }
    cudaEventRecord(e, st);
    ctx->prof_events[kind]->push_back(e);
}

// up to this many histories a block is run by the persistent sweep kernel: its update costs one atomic exchange per visit,
// which loses against a streaming pass over the grid (~12 us at 4 M voxels) once a block has more than ~1e6 visits
constexpr int64_t SMALL_BLOCK_MAX = 4096;
constexpr int64_t DEFAULT_MIN_PLAN_BLOCK = 32768;   // below this a block is too sparse for shared-memory windows

static int g_ctx_count[64];            // live contexts per device (guarded by g_ctx_mu): the last pct_destroy trims the cache
static std::mutex g_ctx_mu;

static double factorial(int k) { double r = 1.0; for (int i = 2; i <= k; ++i) r *= i; return r; }


// rows are only meaningful on the grid and device they were generated for
static bool same_grid(const pct_ctx* ctx, const pct_paths* P) {
    return P->device == ctx->device && P->nx == ctx->geom.nx && P->ny == ctx->geom.ny && P->nz == ctx->geom.nz && P->n_vox == ctx->n_vox;
}

static void free_paths_arrays(pct_paths* P) {
    cudaDeviceSynchronize();         // the buffers go back to the pool on the legacy stream: nothing may still use them
    cache_free(P->N); cache_free(P->start); cache_free(P->end); cache_free(P->ell); cache_free(P->flags); cache_free(P->code_off); cache_free(P->codes);
    if (P->plan) { free_solve_plan(P->plan); P->plan = nullptr; }
    P->N = nullptr; P->start = nullptr; P->end = nullptr; P->ell = nullptr; P->flags = nullptr; P->code_off = nullptr; P->codes = nullptr;
}

static int ensure_ds(pct_ctx* ctx, cudaStream_t st) {
    if (ctx->ds_cap >= ctx->n_vox) return PCT_OK;
    if (ctx->ds) PCT_CUDA(ctx, cudaFree(ctx->ds));
    if (ctx->dsum) PCT_CUDA(ctx, cudaFree(ctx->dsum));
    ctx->ds = nullptr; ctx->dsum = nullptr; ctx->ds_cap = 0;
    PCT_CUDA(ctx, cudaMalloc(&ctx->ds, sizeof(float2) * (size_t)ctx->n_vox));
    PCT_CUDA(ctx, cudaMalloc(&ctx->dsum, sizeof(float) * (size_t)ctx->n_vox));
    ctx->ds_cap = ctx->n_vox;
    PCT_CUDA(ctx, cudaMemsetAsync(ctx->ds, 0, sizeof(float2) * (size_t)ctx->n_vox, st));
    PCT_CUDA(ctx, cudaMemsetAsync(ctx->dsum, 0, sizeof(float) * (size_t)ctx->n_vox, st));
    return PCT_OK;
}

// grow the code stream to hold at least `need` chunks (keeps the first `used` chunks)
static int ensure_codes(pct_ctx* ctx, pct_paths* P, int64_t need, cudaStream_t st) {
    if (need <= P->chunks_cap) return PCT_OK;
    int64_t cap = P->chunks_cap + P->chunks_cap / 2;
    if (cap < need) cap = need;
    ulonglong2* fresh = nullptr;
    cudaError_t e = cache_alloc((void**)&fresh, sizeof(ulonglong2) * (size_t)cap);
    if (e != cudaSuccess && cap > need) { cudaGetLastError(); cap = need; e = cache_alloc((void**)&fresh, sizeof(ulonglong2) * (size_t)cap); }
    if (e != cudaSuccess) { cudaGetLastError(); return set_error(ctx, PCT_E_OOM, "code stream of %lld chunks does not fit", (long long)cap); }
    if (P->chunks_used > 0)
        PCT_CUDA(ctx, cudaMemcpyAsync(fresh, P->codes, sizeof(ulonglong2) * (size_t)P->chunks_used, cudaMemcpyDeviceToDevice, st));
    PCT_CUDA(ctx, cudaStreamSynchronize(st));
    if (P->codes) PCT_CUDA(ctx, cache_free(P->codes));
    P->codes = fresh;
    P->chunks_cap = cap;
    return PCT_OK;
}

}  // namespace pct

namespace pct {
// Before any A1 kernel: the tracker planes of this data set and the clip box of the hull search (find_hull) -- the bounding
// box of the hull voxels, or the grid.  Synchronises `st` when there is a hull.
int prepare_hull_search(pct_ctx* ctx, const pct_protons* pr, const uint8_t* hull, cudaStream_t st) {
    ctx->cfg.u_in = pr->u_in_mm; ctx->cfg.u_out = pr->u_out_mm;
    const int nn[3] = {ctx->geom.nx, ctx->geom.ny, ctx->geom.nz};
    for (int a = 0; a < 3; ++a) { ctx->cfg.bmin[a] = 0; ctx->cfg.bmax[a] = nn[a] - 1; }
    if (hull && pr->m > 0) {
        int box[6];
        int* d_box = reinterpret_cast<int*>(ctx->d_stats);      // scratch of 24 bytes; callers clear d_stats afterwards
        int rc0;
        if ((rc0 = launch_hull_bbox(ctx, hull, d_box, st)) != PCT_OK) return rc0;
        PCT_CUDA(ctx, cudaMemcpyAsync(box, d_box, sizeof(box), cudaMemcpyDeviceToHost, st));
        PCT_CUDA(ctx, cudaStreamSynchronize(st));
        for (int a = 0; a < 3; ++a) {
            if (box[3 + a] >= box[a]) { ctx->cfg.bmin[a] = box[a]; ctx->cfg.bmax[a] = box[3 + a]; }
            else { ctx->cfg.bmin[a] = 0; ctx->cfg.bmax[a] = -1; }               // empty hull: every ray misses
        }
    }
    return PCT_OK;
}

// argument checks shared by the calls that take tracker records
int check_protons(pct_ctx* ctx, const pct_protons* pr) {
    if (!pr || pr->m < 0) return set_error(ctx, PCT_E_INVALID_ARG, "bad protons");
    if (pr->m > 0 && (!pr->phi || !pr->t_in || !pr->v_in || !pr->dt_in || !pr->dv_in || !pr->t_out || !pr->v_out || !pr->dt_out || !pr->dv_out))
        return set_error(ctx, PCT_E_INVALID_ARG, "NULL tracker array");
    if (!std::isfinite(pr->u_in_mm) || !std::isfinite(pr->u_out_mm)) return set_error(ctx, PCT_E_INVALID_ARG, "bad tracker planes");
    return PCT_OK;
}
}  // namespace pct

using namespace pct;

extern "C" {

int pct_create(const pct_geometry* geom, const pct_mlp_params* params, int device, pct_ctx** out) {
    if (!out) return PCT_E_INVALID_ARG;
    *out = nullptr;
    if (!geom || !params) return PCT_E_INVALID_ARG;
    if (geom->nx <= 0 || geom->ny <= 0 || geom->nz <= 0 || !(geom->h_mm > 0.0) || !std::isfinite(geom->h_mm)) return PCT_E_INVALID_ARG;
    if ((int64_t)geom->nx * geom->ny * geom->nz > 0x7fffffffLL) return PCT_E_INVALID_ARG;
    if (!(params->step_frac > 0.0) || !(params->X0_mm > 0.0) || !(params->tie_eps_mm >= 0.0) || params->max_visits < 1 ||
        params->max_visits > MAX_VISITS_LIMIT || !(params->poly_max_depth_mm > 0.0)) return PCT_E_INVALID_ARG;
    for (int i = 0; i < 6; ++i) if (!std::isfinite(params->poly[i])) return PCT_E_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return PCT_E_CUDA; }
    pct_ctx* ctx = new (std::nothrow) pct_ctx();
    if (!ctx) return PCT_E_OOM;
    std::memset(ctx, 0, sizeof(*ctx));
    for (auto& v : ctx->prof_events) v = new std::vector<cudaEvent_t>();
    ctx->prof_pool = new std::vector<cudaEvent_t>();
    ctx->geom = *geom;
    ctx->params = *params;
    ctx->device = device;
    ctx->n_vox = (int64_t)geom->nx * geom->ny * geom->nz;
    ctx->solve_mode = 0;
    ctx->solve_min_block = DEFAULT_MIN_PLAN_BLOCK;
    DevCfg& c = ctx->cfg;
    c.nx = geom->nx; c.ny = geom->ny; c.nz = geom->nz;
    c.sx = 1; c.sy = geom->nx; c.sz = geom->nx * geom->ny;
    c.h = geom->h_mm; c.inv_h = 1.0 / geom->h_mm;
    const int nn[3] = {geom->nx, geom->ny, geom->nz};
    // hi must be bit-identical to the kernels' face_coord(a, n) = fma(n, h, lo): the exit point is snapped to it
    for (int a = 0; a < 3; ++a) { c.lo[a] = geom->origin_mm[a]; c.hi[a] = std::fma((double)nn[a], geom->h_mm, geom->origin_mm[a]); }
    for (int i = 0; i < 6; ++i) {
        c.a[i] = params->poly[i];
        // int_0^W (W-w)^q w^i dw = W^(i+q+1) q! i! / (i+q+1)!
        for (int q = 0; q < 3; ++q) c.s1c[q][i] = params->poly[i] * factorial(q) * factorial(i) / factorial(i + q + 1);
    }
    c.X0 = params->X0_mm; c.log_coeff = params->log_coeff; c.step_frac = params->step_frac;
    c.tie_eps = params->tie_eps_mm; c.max_depth = params->poly_max_depth_mm; c.max_visits = params->max_visits;
    c.stage_chunks = (params->max_visits - 1 + CODES_PER_CHUNK - 1) / CODES_PER_CHUNK;
    if (c.stage_chunks < 1) c.stage_chunks = 1;
    DeviceGuard guard(device);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); pct_destroy(ctx); return PCT_E_CUDA; }
    ctx->num_sms = prop.multiProcessorCount;
    {   // ln k table: K = ceil(D / (step_frac h)) <= ceil(max_depth / (step_frac h)) samples per history (R8)
        const double kmax = std::ceil(params->poly_max_depth_mm / (params->step_frac * geom->h_mm)) + 2.0;
        if (!(kmax < 16.0 * 1024 * 1024)) { pct_destroy(ctx); return PCT_E_INVALID_ARG; }
        ctx->logk_n = (int)kmax + 1;
        std::vector<double> tab((size_t)ctx->logk_n);
        tab[0] = 0.0;
        for (int k = 1; k < ctx->logk_n; ++k) tab[(size_t)k] = std::log((double)k);
        if (cudaMalloc(&ctx->logk, sizeof(double) * tab.size()) != cudaSuccess ||
            cudaMemcpy(ctx->logk, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError(); pct_destroy(ctx); return PCT_E_OOM;
        }
    }
    if (cudaMalloc(&ctx->d_stats, sizeof(GenStats)) != cudaSuccess || cudaMalloc(&ctx->d_total, sizeof(unsigned long long)) != cudaSuccess) {
        cudaGetLastError(); pct_destroy(ctx); return PCT_E_OOM;
    }
    { std::lock_guard<std::mutex> lock(g_ctx_mu); if (device < 64) ++g_ctx_count[device]; ctx->counted = true; }
    *out = ctx;
    return PCT_OK;
}

void pct_destroy(pct_ctx* ctx) {
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    bool last = false;
    if (ctx->counted) { std::lock_guard<std::mutex> lock(g_ctx_mu); if (ctx->device < 64) last = --g_ctx_count[ctx->device] == 0; }
    if (last) cache_trim(ctx->device);
    cudaFree(ctx->ds); cudaFree(ctx->dsum); cudaFree(ctx->counts_buf); cudaFree(ctx->scan_tmp); cudaFree(ctx->logk); cudaFree(ctx->gen_scratch); cudaFree(ctx->d_stats); cudaFree(ctx->d_total);
    for (auto& v : ctx->prof_events) { if (v) { for (cudaEvent_t e : *v) cudaEventDestroy(e); delete v; } }
    if (ctx->prof_pool) { for (cudaEvent_t e : *ctx->prof_pool) cudaEventDestroy(e); delete ctx->prof_pool; }
    delete ctx;
}

int pct_profile_enable(pct_ctx* ctx, int on) {
    if (!ctx) return PCT_E_INVALID_ARG;
    ctx->profiling = on != 0;
    return PCT_OK;
}

int pct_profile_read(pct_ctx* ctx, pct_profile* out) {
    if (!ctx || !out) return PCT_E_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PCT_CUDA(ctx, cudaDeviceSynchronize());
    for (int k = 0; k < PCT_PROFILE_KINDS; ++k) {
        std::vector<cudaEvent_t>& v = *ctx->prof_events[k];
        for (size_t i = 0; i + 1 < v.size(); i += 2) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, v[i], v[i + 1]) == cudaSuccess) { out->ms[k] += ms; out->launches[k] += 1; }
        }
        for (cudaEvent_t e : v) ctx->prof_pool->push_back(e);
        v.clear();
    }
    cudaGetLastError();
    return PCT_OK;
}

const char* pct_last_error(const pct_ctx* ctx) { return ctx ? ctx->err : "null context"; }
int pct_trim_cache(pct_ctx* ctx) {
    if (!ctx) return PCT_E_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    cache_trim(ctx->device);
    return PCT_OK;
}

int64_t pct_launch_count(const pct_ctx* ctx) { return ctx ? ctx->launches : 0; }

int pct_generate_mlp(pct_ctx* ctx, const pct_protons* pr, const uint8_t* hull, void* stream, pct_paths** out) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!out) return set_error(ctx, PCT_E_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!pr || pr->m < 0) return set_error(ctx, PCT_E_INVALID_ARG, "bad protons");
    if (pr->m > 0 && (!pr->phi || !pr->t_in || !pr->v_in || !pr->dt_in || !pr->dv_in || !pr->t_out || !pr->v_out || !pr->dt_out || !pr->dv_out))
        return set_error(ctx, PCT_E_INVALID_ARG, "NULL tracker array");
    if (!std::isfinite(pr->u_in_mm) || !std::isfinite(pr->u_out_mm)) return set_error(ctx, PCT_E_INVALID_ARG, "bad tracker planes");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    {
        const int rc0 = prepare_hull_search(ctx, pr, hull, st);
        if (rc0 != PCT_OK) return rc0;
    }
    pct_paths* P = new (std::nothrow) pct_paths();
    if (!P) return set_error(ctx, PCT_E_OOM, "host allocation");
    std::memset(P, 0, sizeof(*P));
    P->device = ctx->device; P->m = pr->m; P->n_vox = ctx->n_vox;
    P->nx = ctx->geom.nx; P->ny = ctx->geom.ny; P->nz = ctx->geom.nz;
    const int64_t m = pr->m;
    const size_t mm = (size_t)(m > 0 ? m : 1);
    ulonglong2* stage = nullptr;
    int rc = PCT_OK;
    // kernels of this call may still be running on `st`: drain it before any block goes back to the (process-wide) cache
    auto fail = [&](int code) { cudaStreamSynchronize(st); cudaGetLastError(); cache_free(stage); free_paths_arrays(P); delete P; return code; };
#define GEN_CUDA(call)                                                                                          \
    do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError();                               \
        return fail(set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
    GEN_CUDA(cache_alloc((void**)&P->N, sizeof(uint32_t) * mm));
    GEN_CUDA(cache_alloc((void**)&P->start, sizeof(int32_t) * mm));
    GEN_CUDA(cache_alloc((void**)&P->end, sizeof(int32_t) * mm));
    GEN_CUDA(cache_alloc((void**)&P->ell, sizeof(float) * mm));
    GEN_CUDA(cache_alloc((void**)&P->flags, sizeof(uint8_t) * mm));
    GEN_CUDA(cache_alloc((void**)&P->code_off, sizeof(uint64_t) * mm));
    const int batch_max = (int)(m < GEN_BATCH ? (m > 0 ? m : 1) : GEN_BATCH);
    // staging rows of the walk kernel (a row's place in the code stream is known only when its length is)
    GEN_CUDA(cache_alloc((void**)&stage, sizeof(ulonglong2) * (size_t)batch_max * (size_t)ctx->cfg.stage_chunks));
    GEN_CUDA(cudaMemsetAsync(ctx->d_stats, 0, sizeof(GenStats), st));
    // rows are appended to the code stream at places handed out by a device counter (chunks), read back after every batch
    GEN_CUDA(cudaMemsetAsync(ctx->d_total, 0, sizeof(unsigned long long), st));
    const ProtonPtrs pp = {pr->phi, pr->t_in, pr->v_in, pr->dt_in, pr->dv_in, pr->t_out, pr->v_out, pr->dt_out, pr->dv_out};
    for (int64_t i0 = 0; i0 < m; i0 += GEN_BATCH) {
        const int count = (int)((m - i0) < GEN_BATCH ? (m - i0) : GEN_BATCH);
        // room for the worst case of this batch; the first growth extrapolates what the batches so far needed to all histories
        const int64_t reserve = P->chunks_used + (int64_t)count * ctx->cfg.stage_chunks;
        if (reserve > P->chunks_cap) {
            int64_t guess = reserve;
            if (i0 > 0) guess = (int64_t)((double)P->chunks_used * ((double)m / (double)i0) * 1.45) + (int64_t)GEN_BATCH * ctx->cfg.stage_chunks;
            if ((rc = ensure_codes(ctx, P, guess > reserve ? guess : reserve, st)) != PCT_OK) {
                if (!(guess > reserve) || (rc = ensure_codes(ctx, P, reserve, st)) != PCT_OK) return fail(rc);
            }
        }
        if (ctx->batch_ready && i0 / GEN_BATCH < ctx->n_batch_ready) GEN_CUDA(cudaStreamWaitEvent(st, ctx->batch_ready[i0 / GEN_BATCH], 0));
        if ((rc = launch_mlp_batch(ctx, pp, hull, i0, count, stage, ctx->d_total, P, st)) != PCT_OK) return fail(rc);
        unsigned long long used = 0;
        GEN_CUDA(cudaMemcpyAsync(&used, ctx->d_total, sizeof(used), cudaMemcpyDeviceToHost, st));
        GEN_CUDA(cudaStreamSynchronize(st));
        P->chunks_used = (int64_t)used;
    }
    GenStats hs;
    GEN_CUDA(cudaMemcpyAsync(&hs, ctx->d_stats, sizeof(hs), cudaMemcpyDeviceToHost, st));
    GEN_CUDA(cudaStreamSynchronize(st));
#undef GEN_CUDA
    cache_free(stage);
    P->total_visits = (int64_t)hs.total_visits; P->n_rejected = (int64_t)hs.n_rejected; P->total_samples = (int64_t)hs.total_samples; P->n_ties = (int64_t)hs.n_ties; P->n_general = (int64_t)hs.n_general;
    *out = P;
    return PCT_OK;
}

int pct_solve_config(pct_ctx* ctx, int mode, int64_t min_block) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (mode < 0 || mode > 2) return set_error(ctx, PCT_E_INVALID_ARG, "solve mode must be 0, 1 or 2");
    ctx->solve_mode = mode;
    ctx->solve_min_block = min_block > 0 ? min_block : DEFAULT_MIN_PLAN_BLOCK;
    return PCT_OK;
}

int pct_plan_info(const pct_paths* P, pct_plan_stats* out) {
    if (!P || !out) return PCT_E_INVALID_ARG;
    std::memset(out, 0, sizeof(*out));
    const SolvePlan* pl = P->plan;
    if (!pl) return PCT_OK;
    out->block_size = pl->block_size; out->n_blocks = pl->n_blocks; out->n_groups = pl->n_groups; out->n_direct = pl->n_direct;
    // everything the plan keeps resident: visit counts, code stream, perm + p0 + pflag + direct list (13 bytes per history),
    // group table, launch order, per-block direct counts
    out->plan_bytes = pl->cnt_bytes + 8 * pl->stream_words + P->m * 13 + (pl->n_groups + 1) * (int64_t)sizeof(PlanGroup) + pl->n_groups * 4 + pl->n_blocks * 4;
    out->stream_bytes = 8 * pl->stream_words; out->cnt_bytes = pl->cnt_bytes;
    out->staged_slots = pl->staged_slots; out->windowed_histories = pl->windowed_histories; out->windowed_visits = pl->windowed_visits;
    return PCT_OK;
}

int pct_paths_info(const pct_paths* P, pct_paths_stats* out) {
    if (!P || !out) return PCT_E_INVALID_ARG;
    out->m = P->m; out->total_visits = P->total_visits; out->n_rejected = P->n_rejected; out->n_ties = P->n_ties;
    out->total_samples = P->total_samples; out->n_general_segments = P->n_general;
    out->code_bytes = P->chunks_used * (int64_t)sizeof(ulonglong2);
    out->header_bytes = P->m * (int64_t)(sizeof(uint32_t) + 2 * sizeof(int32_t) + sizeof(float) + sizeof(uint8_t) + sizeof(uint64_t));
    return PCT_OK;
}

void pct_paths_free(pct_paths* P) {
    if (!P) return;
    DeviceGuard guard(P->device);
    free_paths_arrays(P);
    delete P;
}

int pct_paths_decode(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, int64_t* row_ptr, int32_t* voxels, int64_t cap,
                     float* ell, uint8_t* flags, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!P || !row_ptr || i0 < 0 || i1 > P->m || i0 > i1) return set_error(ctx, PCT_E_INVALID_ARG, "bad decode range");
    if (!same_grid(ctx, P)) return set_error(ctx, PCT_E_INVALID_ARG, "paths were generated on another grid or device");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t cnt = i1 - i0;
    int rc;
    if ((rc = launch_scan_u32(ctx, P->N + i0, (uint64_t*)row_ptr, cnt, 0, ctx->d_total, st)) != PCT_OK) return rc;
    PCT_CUDA(ctx, cudaMemcpyAsync(row_ptr + cnt, ctx->d_total, sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
    unsigned long long total = 0;
    PCT_CUDA(ctx, cudaMemcpyAsync(&total, ctx->d_total, sizeof(total), cudaMemcpyDeviceToHost, st));
    if (ell && cnt) PCT_CUDA(ctx, cudaMemcpyAsync(ell, P->ell + i0, sizeof(float) * (size_t)cnt, cudaMemcpyDeviceToDevice, st));
    if (flags && cnt) PCT_CUDA(ctx, cudaMemcpyAsync(flags, P->flags + i0, (size_t)cnt, cudaMemcpyDeviceToDevice, st));
    PCT_CUDA(ctx, cudaStreamSynchronize(st));
    if (voxels) {
        if ((int64_t)total > cap) return set_error(ctx, PCT_E_CAPACITY, "decode needs %llu voxel slots, cap is %lld", total, (long long)cap);
        if ((rc = launch_decode(ctx, P, i0, i1, (const uint64_t*)row_ptr, voxels, st)) != PCT_OK) return rc;
        PCT_CUDA(ctx, cudaStreamSynchronize(st));
    }
    return PCT_OK;
}

int pct_paths_flagged(pct_ctx* ctx, const pct_paths* P, uint32_t mask, int64_t* idx_out, int64_t cap, int64_t* n_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!P || !n_out || cap < 0 || (cap > 0 && !idx_out)) return set_error(ctx, PCT_E_INVALID_ARG, "bad flagged-list arguments");
    if (!same_grid(ctx, P)) return set_error(ctx, PCT_E_INVALID_ARG, "paths were generated on another grid or device");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    *n_out = 0;
    if (P->m == 0) return PCT_OK;
    uint32_t* d_idx = nullptr;
    const int64_t keep = cap < P->m ? cap : P->m;
    PCT_CUDA(ctx, cache_alloc((void**)&d_idx, sizeof(uint32_t) * (size_t)(keep > 0 ? keep : 1)));
    int rc = launch_collect_flagged(ctx, P, mask, d_idx, keep, ctx->d_total, st);
    unsigned long long n = 0;
    std::vector<uint32_t> host((size_t)keep);
    cudaError_t e = rc == PCT_OK ? cudaMemcpyAsync(&n, ctx->d_total, sizeof(n), cudaMemcpyDeviceToHost, st) : cudaSuccess;
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    const int64_t got = (int64_t)n < keep ? (int64_t)n : keep;
    if (e == cudaSuccess && got > 0) e = cudaMemcpy(host.data(), d_idx, sizeof(uint32_t) * (size_t)got, cudaMemcpyDeviceToHost);
    cudaStreamSynchronize(st);
    cache_free(d_idx);
    if (rc != PCT_OK) return rc;
    if (e != cudaSuccess) { cudaGetLastError(); return set_error(ctx, PCT_E_CUDA, "flagged list: %s", cudaGetErrorString(e)); }
    std::sort(host.begin(), host.begin() + got);
    for (int64_t k = 0; k < got; ++k) idx_out[k] = (int64_t)host[(size_t)k];
    *n_out = (int64_t)n;
    return PCT_OK;
}

int pct_forward_project(pct_ctx* ctx, const pct_paths* P, const float* x, float* b_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!P || !x || (!b_out && P->m > 0)) return set_error(ctx, PCT_E_INVALID_ARG, "bad forward_project arguments");
    if (!same_grid(ctx, P)) return set_error(ctx, PCT_E_INVALID_ARG, "paths were generated on another grid or device");
    DeviceGuard guard(ctx->device);
    return launch_forward_project(ctx, P, x, b_out, (cudaStream_t)stream);
}

int pct_column_counts(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, uint32_t* counts, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!P || !counts || i0 < 0 || i1 > P->m || i0 > i1) return set_error(ctx, PCT_E_INVALID_ARG, "bad column_counts arguments");
    if (!same_grid(ctx, P)) return set_error(ctx, PCT_E_INVALID_ARG, "paths were generated on another grid or device");
    DeviceGuard guard(ctx->device);
    return launch_column_counts(ctx, P, i0, i1, counts, (cudaStream_t)stream);
}

// A8: the iteration driver.  iters x ceil(m/B) x (project+scatter, update) on one stream, no host sync inside.
int pct_solve(pct_ctx* ctx, pct_paths* P, const float* b, const float* x0, int iters, int64_t block_size, float lambda,
              float* x_out, void* stream) {
    return pct_solve_ex(ctx, P, b, x0, iters, block_size, lambda, nullptr, x_out, stream);
}

int pct_solve_ex(pct_ctx* ctx, pct_paths* P, const float* b, const float* x0, int iters, int64_t block_size, float lambda,
                 const pct_solve_opts* opts, float* x_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    const float* wts = opts ? opts->weights : nullptr;
    const float clamp_lo = opts ? opts->clamp_lo : 1.f, clamp_hi = opts ? opts->clamp_hi : 0.f;       // lo > hi: no clamp
    if (opts && (std::isnan(opts->clamp_lo) || std::isnan(opts->clamp_hi))) return set_error(ctx, PCT_E_INVALID_ARG, "NaN clamp bound");
    if (!P || (!b && P->m > 0) || !x0 || !x_out || iters < 0 || block_size < 1 || !std::isfinite(lambda))
        return set_error(ctx, PCT_E_INVALID_ARG, "bad solve arguments");
    if (!same_grid(ctx, P)) return set_error(ctx, PCT_E_INVALID_ARG, "paths were generated on another grid or device");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if ((rc = ensure_ds(ctx, st)) != PCT_OK) return rc;
    if (x_out != x0) PCT_CUDA(ctx, cudaMemcpyAsync(x_out, x0, sizeof(float) * (size_t)ctx->n_vox, cudaMemcpyDeviceToDevice, st));
    // the plan is built once per (paths, block_size) and cached in the paths object
    const SolvePlan* plan = nullptr;
    const int64_t n_blocks = P->m > 0 ? (P->m + block_size - 1) / block_size : 0;
    const bool plan_possible = iters > 0 && P->m > 0 && P->m < 0xffffffffLL && n_blocks < (1LL << 24);
    const bool want_plan = ctx->solve_mode == 2 || (ctx->solve_mode == 0 && (P->m < block_size ? P->m : block_size) >= ctx->solve_min_block);
    if (plan_possible && want_plan) {
        pct_paths* Pm = P;
        if (Pm->plan && Pm->plan->block_size != block_size) { free_solve_plan(Pm->plan); Pm->plan = nullptr; }
        if (!Pm->plan) {
            ProfScope prof(ctx, 4, st);
            rc = build_solve_plan(ctx, P, block_size, st, &Pm->plan);
            if (rc == PCT_E_OOM) { Pm->plan = nullptr; cudaGetLastError(); }      // no room for the plan: direct kernels
            else if (rc != PCT_OK) return rc;
        }
        plan = Pm->plan;
    }
    // count cache (R23): one buffer per context, owned by the plan that filled it last
    uint32_t* plan_counts = nullptr;
    if (plan) {
        // n_blocks x n_vox counts, then 8 ints per block: the bounding box of the voxels the block visits
        const size_t need = 4 * (size_t)plan->n_blocks * (size_t)ctx->n_vox + 32 * (size_t)plan->n_blocks;
        if (need > ctx->counts_cap) {
            size_t free_b = 0, total_b = 0;
            if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && need <= (free_b + ctx->counts_cap) / 4 && need <= ((size_t)32 << 30)) {
                PCT_CUDA(ctx, cudaStreamSynchronize(st));
                cudaFree(ctx->counts_buf);
                ctx->counts_buf = nullptr; ctx->counts_cap = 0; ctx->counts_owner = nullptr;
                if (cudaMalloc(&ctx->counts_buf, need) == cudaSuccess) ctx->counts_cap = need;
                else cudaGetLastError();
            }
        }
        if (need <= ctx->counts_cap) {
            if (ctx->counts_owner != plan) {
                std::fill(const_cast<SolvePlan*>(plan)->counts_ready.begin(), const_cast<SolvePlan*>(plan)->counts_ready.end(), (uint8_t)0);
                ctx->counts_owner = plan;
            }
            plan_counts = ctx->counts_buf;
        }
    }
    // small blocks on the direct path: all sweeps in one persistent cooperative kernel (solve_kernels.cu); PCT_HOST_SWEEPS=1
    // keeps the launch-per-block loop (A/B, debugging)
    if (!plan && n_blocks >= 4 && block_size <= SMALL_BLOCK_MAX && !getenv("PCT_HOST_SWEEPS")) {
        rc = launch_sweeps_persistent(ctx, P, b, wts, x_out, iters, block_size, lambda, clamp_lo, clamp_hi, st);
        if (rc != PCT_E_CAPACITY) return rc;
    }
    for (int it = 0; it < iters; ++it) {
        for (int64_t t = 0, i0 = 0; i0 < P->m; i0 += block_size, ++t) {
            const int64_t i1 = (P->m - i0) < block_size ? P->m : i0 + block_size;
            if (plan) {
                // s_j^t does not depend on x (R15): the first sweep over block t counts and stores it, later sweeps
                // (and later calls with the same paths and block size) accumulate Delta only
                uint32_t* counts = plan_counts ? plan_counts + (size_t)t * (size_t)ctx->n_vox : nullptr;
                const bool cached = counts && plan->counts_ready[(size_t)t];
                int* box6 = counts ? reinterpret_cast<int*>(plan_counts + (size_t)plan->n_blocks * (size_t)ctx->n_vox) + 8 * t : nullptr;
                if ((rc = launch_block_windowed(ctx, P, plan, t, !cached, b, wts, x_out, ctx->ds, ctx->dsum, st)) != PCT_OK) return rc;
                const int64_t nd = plan->direct_count[(size_t)t];
                if (nd > 0 && (rc = launch_block_project_scatter(ctx, P, i0, i0 + nd, plan->direct_list, !cached, b, wts, x_out, ctx->ds, ctx->dsum, st)) != PCT_OK) return rc;
                if ((rc = launch_block_update(ctx, x_out, ctx->ds, ctx->dsum, counts, !cached, lambda, clamp_lo, clamp_hi, box6, st)) != PCT_OK) return rc;
                if (counts) const_cast<SolvePlan*>(plan)->counts_ready[(size_t)t] = 1;
            } else {
                if ((rc = launch_block_project_scatter(ctx, P, i0, i1, nullptr, true, b, wts, x_out, ctx->ds, ctx->dsum, st)) != PCT_OK) return rc;
                if ((rc = launch_block_update(ctx, x_out, ctx->ds, ctx->dsum, nullptr, false, lambda, clamp_lo, clamp_hi, nullptr, st)) != PCT_OK) return rc;
            }
        }
    }
    return PCT_OK;
}

int pct_reconstruct_host(pct_ctx* ctx, const pct_protons* pr, const uint8_t* hull_host, const float* b_host, const float* x0_host,
                         int iters, int64_t block_size, float lambda, float* x_out_host, pct_recon_stats* stats, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!pr || pr->m < 0 || !b_host || !x_out_host || iters < 0 || block_size < 1) return set_error(ctx, PCT_E_INVALID_ARG, "bad reconstruct arguments");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t m = pr->m, n = ctx->n_vox;
    const size_t mm = (size_t)(m > 0 ? m : 1);
    double* d_tr = nullptr; float* d_b = nullptr; float* d_x = nullptr; uint8_t* d_hull = nullptr;
    pct_paths* P = nullptr;
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    // the tracker arrays travel on a copy stream, one generation batch at a time, while K1 works on the batches that
    // have arrived; b follows them and is awaited before the solve
    cudaStream_t cs = nullptr;
    cudaEvent_t ev_alloc = nullptr, ev_c0 = nullptr, ev_c1 = nullptr;
    const int n_batches = (int)((m + GEN_BATCH - 1) / GEN_BATCH);
    std::vector<cudaEvent_t> ready((size_t)n_batches, nullptr);
    int rc = PCT_OK;
    auto cleanup = [&]() {
        ctx->batch_ready = nullptr; ctx->n_batch_ready = 0;
        // on the error paths kernels and copies may still be in flight: nothing returns to the cache before both streams drain
        cudaStreamSynchronize(st);
        if (cs) cudaStreamSynchronize(cs);
        cudaGetLastError();
        cache_free(d_tr); cache_free(d_b); cache_free(d_x); cache_free(d_hull);
        if (P) pct_paths_free(P);
        for (auto& e : ev) if (e) cudaEventDestroy(e);
        for (auto& e : ready) if (e) cudaEventDestroy(e);
        if (ev_alloc) cudaEventDestroy(ev_alloc);
        if (ev_c0) cudaEventDestroy(ev_c0);
        if (ev_c1) cudaEventDestroy(ev_c1);
        if (cs) cudaStreamDestroy(cs);
    };
#define REC_CUDA(call)                                                                                          \
    do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError(); cleanup();                    \
        return set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__)); } } while (0)
    const bool dbg = getenv("PCT_PLAN_DEBUG") != nullptr;
    const auto t_begin = std::chrono::steady_clock::now();
    auto stamp = [&](const char* what) {
        if (dbg) fprintf(stderr, "[recon] %-22s at %8.2f ms\n", what, std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count());
    };
    for (auto& e : ev) REC_CUDA(cudaEventCreate(&e));
    REC_CUDA(cache_alloc((void**)&d_tr, sizeof(double) * 9 * mm));
    REC_CUDA(cache_alloc((void**)&d_b, sizeof(float) * mm));
    REC_CUDA(cache_alloc((void**)&d_x, sizeof(float) * (size_t)n));
    if (hull_host) REC_CUDA(cache_alloc((void**)&d_hull, (size_t)n));
    stamp("allocated");
    REC_CUDA(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    REC_CUDA(cudaEventCreateWithFlags(&ev_alloc, cudaEventDisableTiming));
    REC_CUDA(cudaEventCreate(&ev_c0));
    REC_CUDA(cudaEventCreate(&ev_c1));
    for (auto& e : ready) REC_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    REC_CUDA(cudaEventRecord(ev[0], st));
    REC_CUDA(cudaEventRecord(ev_alloc, st));
    REC_CUDA(cudaStreamWaitEvent(cs, ev_alloc, 0));          // the copy stream starts behind whatever `st` still runs on these (reused) blocks
    // small inputs first: the copy engine serves requests in issue order, and K1 needs the hull before its first batch
    if (hull_host) REC_CUDA(cudaMemcpyAsync(d_hull, hull_host, (size_t)n, cudaMemcpyHostToDevice, st));
    if (x0_host) REC_CUDA(cudaMemcpyAsync(d_x, x0_host, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, st));
    REC_CUDA(cudaEventRecord(ev[1], st));
    REC_CUDA(cudaEventRecord(ev_c0, cs));
    const double* src[9] = {pr->phi, pr->t_in, pr->v_in, pr->dt_in, pr->dv_in, pr->t_out, pr->v_out, pr->dt_out, pr->dv_out};
    for (int bi = 0; bi < n_batches; ++bi) {
        const int64_t i0 = (int64_t)bi * GEN_BATCH;
        const size_t cnt = (size_t)((m - i0) < GEN_BATCH ? (m - i0) : GEN_BATCH);
        for (int k = 0; k < 9; ++k)
            REC_CUDA(cudaMemcpyAsync(d_tr + (size_t)k * mm + i0, src[k] + i0, sizeof(double) * cnt, cudaMemcpyHostToDevice, cs));
        REC_CUDA(cudaEventRecord(ready[(size_t)bi], cs));
    }
    if (m > 0) REC_CUDA(cudaMemcpyAsync(d_b, b_host, sizeof(float) * (size_t)m, cudaMemcpyHostToDevice, cs));
    REC_CUDA(cudaEventRecord(ev_c1, cs));
    pct_protons dev = *pr;
    dev.phi = d_tr; dev.t_in = d_tr + mm; dev.v_in = d_tr + 2 * mm; dev.dt_in = d_tr + 3 * mm; dev.dv_in = d_tr + 4 * mm;
    dev.t_out = d_tr + 5 * mm; dev.v_out = d_tr + 6 * mm; dev.dt_out = d_tr + 7 * mm; dev.dv_out = d_tr + 8 * mm;
    stamp("copies enqueued");
    ctx->batch_ready = ready.data(); ctx->n_batch_ready = n_batches;
    rc = pct_generate_mlp(ctx, &dev, d_hull, stream, &P);
    ctx->batch_ready = nullptr; ctx->n_batch_ready = 0;
    if (rc != PCT_OK) { cleanup(); return rc; }
    REC_CUDA(cudaEventRecord(ev[2], st));
    stamp("generate returned");
    REC_CUDA(cudaStreamWaitEvent(st, ev_c1, 0));              // b has arrived
    if (!x0_host && (rc = launch_fill(ctx, d_x, n, 1.0f, st)) != PCT_OK) { cleanup(); return rc; }   // x0 = 1 (BASELINE.json configs)
    if ((rc = pct_solve(ctx, P, d_b, d_x, iters, block_size, lambda, d_x, stream)) != PCT_OK) { cleanup(); return rc; }
    REC_CUDA(cudaEventRecord(ev[3], st));
    REC_CUDA(cudaMemcpyAsync(x_out_host, d_x, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, st));
    REC_CUDA(cudaEventRecord(ev[4], st));
    stamp("solve enqueued");
    REC_CUDA(cudaStreamSynchronize(st));
    stamp("stream drained");
    if (stats) {
        stats->m = m; stats->total_visits = P->total_visits; stats->n_rejected = P->n_rejected; stats->n_ties = P->n_ties;
        float ms[4] = {0, 0, 0, 0};
        for (int k = 0; k < 4; ++k) cudaEventElapsedTime(&ms[k], ev[k], ev[k + 1]);
        cudaEventElapsedTime(&ms[0], ev_c0, ev_c1);          // span of the copy stream; it overlaps ms_mlp
        stats->ms_h2d = ms[0]; stats->ms_mlp = ms[1]; stats->ms_solve = ms[2]; stats->ms_d2h = ms[3];
    }
#undef REC_CUDA
    cleanup();
    stamp("cleaned up");
    return PCT_OK;
}

}  // extern "C"
