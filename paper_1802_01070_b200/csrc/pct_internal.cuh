// pct_internal.cuh -- shared declarations of libpct.so (CUDA path only; nothing here is used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "pct.h"

namespace pct {

// ---- encoding of one row of A (R9-R12) -------------------------------------------------------------------
// A row is  start voxel (int32)  +  N-1 face-step codes of 3 bits:  0:+x 1:-x 2:+y 3:-y 4:+z 5:-z 7:pad.
// Codes are packed 21 per uint64 (bits 3k..3k+2), two uint64 = one 16-byte chunk = 42 codes, so the stream is
// read with 128-bit loads and every row starts on a 16-byte boundary.
constexpr int CODES_PER_WORD = 21;
constexpr int CODES_PER_CHUNK = 42;
constexpr int MAX_VISITS_LIMIT = 8192;
constexpr int GEN_BATCH = 1 << 20;   // histories per generation batch (bounds the worst-case staging buffer)

// constants handed to kernels by value (__grid_constant__)
struct DevCfg {
    int nx, ny, nz;
    int sx, sy, sz;            // linear strides 1, nx, nx*ny
    double h, inv_h;
    double lo[3], hi[3];
    double a[6];               // f(w) = sum a_i w^i
    double s1c[3][6];          // Sigma1 moments: I_q(w) = w^(q+1) * sum_i s1c[q][i] w^i,  s1c[q][i] = a_i q! i!/(i+q+1)!
    double X0, log_coeff, step_frac, tie_eps, max_depth;
    int max_visits;
    int stage_chunks;          // chunks of the longest possible row (max_visits)
    double u_in, u_out;
    int bmin[3], bmax[3];      // bounding box of the hull voxels (inclusive); the whole grid if hull == NULL
};

struct ProtonPtrs {
    const double *phi, *t_in, *v_in, *dt_in, *dv_in, *t_out, *v_out, *dt_out, *dv_out;
};

struct GenStats { unsigned long long total_visits, n_rejected, n_ties, total_samples, n_general; };

// ---- solve plan: a block's histories regrouped into spatially compact tubes ----------------------
// A group = up to GROUP histories of one block that travel the same way (class = major axis and direction) and lie
// next to each other.  Row r of a group is the grid plane  major index = m_first + dir*r ; in that row the group's
// window covers WIN_N voxels of the minor in-plane axis from nbase(r) and WIN_Z slices from zbase(r), where the bases
// drift linearly with r (16.16 fixed point).  Window slots are addressed circularly (coordinate mod window size), so a
// history walking its codes needs no knowledge of the bases.  SLAB rows are resident in shared memory at a time.
constexpr int WIN_N = 32, WIN_Z = 16, SLAB = 16;
constexpr int WIN_SLOTS = WIN_N * WIN_Z * SLAB;            // 8192
constexpr int GROUP = 1024;                                // histories per group = threads per CTA
constexpr int MAX_ROW_VISITS = 6;                          // verified per history and row; bounds the fixed-point sums
constexpr int ZROW = 4;                                    // sort rows: slices per z-row of the reference plane

struct PlanGroup {
    uint32_t start;      // first position in perm
    uint32_t size;       // histories in the group (<= GROUP)
    int32_t cls;         // travel code of the group: 0:+x 1:-x 2:+y 3:-y
    int32_t nslab;       // slabs of SLAB rows
    int32_t m_first;     // major-axis index of row 0
    int32_t nb0, zb0;    // window base at row 0 (minor in-plane axis, z), 16.16 fixed point
    int32_t sn, sz;      // base drift per row, 16.16 fixed point
    int32_t wps;         // 64-bit code words per (slab, thread) in the group's slab-aligned code stream
    uint64_t cnt_off;    // first byte of this group's visits-per-slab table: cnt[cnt_off + slab*GROUP + thread]
    uint64_t stream_off; // first word of the group's code stream: stream[stream_off + (slab*wps + w)*GROUP + thread]
    // part of the window the verified members actually visit, as offsets from the row's window base (k_plan_walk):
    // n - nbase(r) in [dn_lo, dn_hi], z - zbase(r) in [dz_lo, dz_hi].  Only that part is staged and flushed.
    int32_t dn_lo, dn_hi, dz_lo, dz_hi;
    int32_t max_cnt;     // largest number of visits one window slot of this group receives in a slab, measured by the first
                         // (counting) sweep; 0 = not measured yet.  Bounds the additions per slot of the fixed-point Delta.
};

// thread -> rank of its history in the group's sorted order.  Transposed on purpose: the lanes of a warp take
// histories spread over the whole cross-section of the tube, so that they rarely hit the same window slot at once.
__host__ __device__ __forceinline__ int plan_rank(int tid, int size) {
    const int warps = (size + 31) >> 5;
    const int w = tid >> 5;
    if (w >= warps) return -1;
    const int rk = (tid & 31) * warps + w;
    return rk < size ? rk : -1;
}
constexpr int PLAN_CODE_FIRST = 6;   // slab stream: "visit here, no step" (the first visit of a history); 7 = pad

__host__ __device__ __forceinline__ int plan_nbase(const PlanGroup& g, int r) { return (int)(((long long)g.nb0 + (long long)r * g.sn) >> 16); }
__host__ __device__ __forceinline__ int plan_zbase(const PlanGroup& g, int r) { return (int)(((long long)g.zb0 + (long long)r * g.sz) >> 16); }

// Packed window coordinate of a visit = byte offset of its 4-byte slot: (n mod 32) << 2 | (row mod 16) << 7 |
// (z mod 16) << 11.  The shared-memory address XORs the row and the low bit of z into the n field (one shift, one LOP3): the lanes of a
// warp sit in the same few rows but in different (n, z) columns of the tube, so the bank must depend on n AND z.
__host__ __device__ __forceinline__ unsigned win_pack(int n, int r, int z) {
    return ((unsigned)(n & (WIN_N - 1)) << 2) | ((unsigned)(r & (SLAB - 1)) << 7) | ((unsigned)(z & (WIN_Z - 1)) << 11);
}
__host__ __device__ __forceinline__ unsigned win_addr(unsigned p) { return p ^ ((p >> 5) & 0x7Cu); }

struct SolvePlan {
    int64_t block_size, n_blocks, n_groups, n_direct, cnt_bytes;
    int64_t staged_slots, windowed_histories, windowed_visits;   // per sweep (pct_plan_info)
    uint32_t* perm;          // sorted position -> history index (m)
    uint32_t* p0;            // packed window coordinate of the first visit, per sorted position
    uint8_t* pflag;          // per sorted position: 1 = windowed, 0 = not (rejected, or listed in direct_list)
    uint8_t* cnt;            // visits per (group, slab, thread)
    std::vector<uint8_t> counts_ready;   // per block (host): s^t of that block is in the context's count cache
    unsigned long long* stream;   // slab-aligned copy of the windowed histories' codes (21 codes per word)
    int64_t stream_words;
    PlanGroup* groups;
    uint32_t* launch_order;  // CTA -> group: a block's groups in order of decreasing work (longest first, shorter tail)
    uint32_t* direct_list;   // histories that take the direct path; block t owns [t*block_size, t*block_size + direct_count[t])
    uint32_t* d_direct_count;
    std::vector<int64_t> group_begin;    // per block, + sentinel (host)
    std::vector<uint32_t> direct_count;  // per block (host)
};

}  // namespace pct

struct pct_ctx {
    pct_geometry geom;
    pct_mlp_params params;
    pct::DevCfg cfg;
    int device;
    int num_sms;
    int64_t n_vox;
    int64_t launches;
    char err[512];
    // scratch owned by the context (grown on demand)
    int solve_mode;      // 0 auto, 1 direct kernel only, 2 windowed plan whenever possible (pct_solve_config)
    int64_t solve_min_block;  // auto: blocks smaller than this take the direct kernel
    float2* ds;          // {Delta_j, s_j} accumulator, n_vox
    uint32_t* counts_buf;     // cache of s_j^t, n_blocks x n_vox, of the plan `counts_owner` (one buffer per context, grown
    size_t counts_cap;        // on demand and kept: a multi-GB allocation per reconstruction is not free)
    const void* counts_owner;
    float* dsum;         // Delta_j accumulator used when the block's counts are cached, n_vox
    int64_t ds_cap;
    void* scan_tmp;      // block sums for scans
    int64_t scan_tmp_bytes;
    cudaEvent_t* batch_ready;   // pct_reconstruct_host: event b = tracker data of generation batch b has arrived (else NULL)
    int n_batch_ready;
    void* gen_scratch;   // pct_generate_mlp: hull records + sort buffers of one batch
    size_t gen_scratch_bytes;
    double* logk;        // ln k for k = 0..logk_n-1 (k = 0 unused): the MLP's two log terms are ln(k du / X0), R8
    int logk_n;
    pct::GenStats* d_stats;
    unsigned long long* d_total;
    // optional per-kernel event timing (pct_profile_enable)
    bool profiling;
    std::vector<cudaEvent_t>* prof_events[PCT_PROFILE_KINDS];   // start/stop pairs per kind
    std::vector<cudaEvent_t>* prof_pool;   // recycled events
    bool k2w_ready;      // dynamic shared memory attribute of k_block_windowed set on this device
    bool counted;        // this context is in the per-device count of live contexts (pct_create completed)
};

struct pct_paths {
    int device;
    int nx, ny, nz;      // grid the rows were generated on: every later call checks its context against them
    int64_t m, n_vox;
    uint32_t* N;         // path entries per history
    int32_t* start;      // start voxel
    float* ell;          // mean chord l_i (R11)
    uint8_t* flags;
    int32_t* end;        // voxel the walk ended in (R10); used by the solve plan only
    uint64_t* code_off;  // first 16-byte chunk of the row in `codes`
    ulonglong2* codes;
    int64_t chunks_used, chunks_cap;
    int64_t total_visits, n_rejected, n_ties, total_samples, n_general;
    pct::SolvePlan* plan; // cached by pct_solve for (this, block_size); owned by the paths object
};

namespace pct {

int set_error(pct_ctx* ctx, int code, const char* fmt, ...);

// Large, short-lived buffers (paths, plans, sort scratch) come from a size-keyed cache of device blocks (pct_api.cu).
cudaError_t cache_alloc(void** p, size_t bytes);
cudaError_t cache_free(void* p);
void cache_trim(int device);

// RAII bracket around one kernel launch when profiling is on (kinds: pct.h, pct_profile)
struct ProfScope {
    pct_ctx* ctx; int kind; cudaStream_t st; bool on;
    ProfScope(pct_ctx* c, int k, cudaStream_t s);
    ~ProfScope();
};

#define PCT_CUDA(ctx, call)                                                                              \
    do {                                                                                                 \
        cudaError_t e__ = (call);                                                                        \
        if (e__ != cudaSuccess)                                                                          \
            return pct::set_error((ctx), e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA,      \
                                  "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

// makes `dev` current for the scope of a call
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int prepare_hull_search(pct_ctx* ctx, const pct_protons* pr, const uint8_t* hull, cudaStream_t st);
int check_protons(pct_ctx* ctx, const pct_protons* pr);
int launch_hull_batch(pct_ctx* ctx, const ProtonPtrs& pr, const uint8_t* hull, int64_t i_base, int count, int32_t* v_in, int32_t* v_out, cudaStream_t st);

// launchers implemented in the .cu files (all enqueue on `st`, none synchronises unless stated)
int launch_mlp_batch(pct_ctx* ctx, const ProtonPtrs& pr, const uint8_t* hull, int64_t i_base, int count, ulonglong2* stage,
                     unsigned long long* chunk_counter, pct_paths* P, cudaStream_t st);
int launch_hull_bbox(pct_ctx* ctx, const uint8_t* hull, int* d_box6, cudaStream_t st);
int launch_scan_u32(pct_ctx* ctx, const uint32_t* in, uint64_t* out, int64_t n, uint64_t base,
                    unsigned long long* d_total, cudaStream_t st);
int launch_decode(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, const uint64_t* row_ptr, int32_t* voxels,
                  cudaStream_t st);
int launch_forward_project(pct_ctx* ctx, const pct_paths* P, const float* x, float* b_out, cudaStream_t st);
int launch_column_counts(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, uint32_t* counts, cudaStream_t st);
int launch_block_project_scatter(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, const uint32_t* list, bool count,
                                 const float* b, const float* wts, const float* x, float2* ds, float* dsum, cudaStream_t st);
int launch_block_windowed(pct_ctx* ctx, const pct_paths* P, const SolvePlan* plan, int64_t block, bool count, const float* b,
                          const float* wts, const float* x, float2* ds, float* dsum, cudaStream_t st);
int build_solve_plan(pct_ctx* ctx, const pct_paths* P, int64_t block_size, cudaStream_t st, SolvePlan** out);
void free_solve_plan(SolvePlan* plan);
int launch_block_update(pct_ctx* ctx, float* x, float2* ds, float* dsum, uint32_t* counts, bool store, float lambda, float clamp_lo,
                        float clamp_hi, int* box6, cudaStream_t st);
int launch_fill(pct_ctx* ctx, float* p, int64_t n, float value, cudaStream_t st);
int launch_sweeps_persistent(pct_ctx* ctx, const pct_paths* P, const float* b, const float* wts, float* x, int iters, int64_t block_size, float lambda,
                        float clamp_lo, float clamp_hi, cudaStream_t st);
int launch_collect_flagged(pct_ctx* ctx, const pct_paths* P, unsigned mask, uint32_t* idx, int64_t cap, unsigned long long* d_count, cudaStream_t st);

}  // namespace pct
