// plan.cu -- the solve plan: regroups every block's histories into spatially compact "tubes" so that
// the block projection (A5/A6, "the block size is the number of protons to be processed in parallel")
// can gather x and accumulate {Delta, s} in shared memory instead of L2.
//
// Reading R18/R22: inside a block the update is simultaneous, so the order in which a block's histories are
// processed is free; block membership (R13, consecutive input ranges) is never changed.
//
// Steps (all on the device, one host synchronisation at the end to read the per-block group ranges):
//   1. k_plan_keys      key_i = (block, travel class, z-row, lateral position at the grid's mid plane) from the start
//                       and end voxel of the row; rejected histories get class 7 (sorted last in their block).
//   2. radix sort       (key, i) pairs -- cub::DeviceRadixSort, the one library primitive used (a plain sort).
//   3. k_plan_heads     group heads: every change of (block, class, z-row) and every GROUP-th sorted position.
//   4. k_plan_params    per group: travel class, first row, window centre line (weighted mean of its members).
//   5. k_plan_walk      WALKS THE CODES of every member once: checks that each visit lies inside the group's window,
//                       that the history never steps against the travel direction, never has more than MAX_ROW_VISITS
//                       visits in one row nor more than the slab's word budget (fixed from the tube's slope in step 4);
//                       records visits per slab and the packed start coordinate; re-emits the codes slab-aligned.
//                       A history that fails is appended to its block's direct list.
// Correctness of the solver never depends on the sort or the centre-line fit: a history is either verified to stay
// in its group's window or it takes the direct kernel.
#include <chrono>
#include <cstdio>
#include <cstdlib>

#include <cub/device/device_radix_sort.cuh>

#include "pct_internal.cuh"

namespace pct {

constexpr int KEY_NREF_BITS = 24, KEY_ZROW_BITS = 13, KEY_CLS_BITS = 3;
constexpr int KEY_RUN_SHIFT = KEY_NREF_BITS;                                   // bits above = (block, class, z-row)
constexpr int KEY_BLOCK_SHIFT = KEY_NREF_BITS + KEY_ZROW_BITS + KEY_CLS_BITS;   // 40

struct ChordInfo { int cls; int m_s, m_e, n_s, n_e, z_s, z_e; };

// start/end voxel -> travel class and (major, minor, z) coordinates of both ends
__device__ __forceinline__ ChordInfo chord_info(const DevCfg& g, int start, int end) {
    ChordInfo c;
    const int sx = start % g.nx, sy = (start / g.nx) % g.ny, sz = start / (g.nx * g.ny);
    const int ex = end % g.nx, ey = (end / g.nx) % g.ny, ez = end / (g.nx * g.ny);
    const int dx = ex - sx, dy = ey - sy;
    if (abs(dx) >= abs(dy)) { c.cls = dx >= 0 ? 0 : 1; c.m_s = sx; c.m_e = ex; c.n_s = sy; c.n_e = ey; }
    else { c.cls = dy >= 0 ? 2 : 3; c.m_s = sy; c.m_e = ey; c.n_s = sx; c.n_e = ex; }
    c.z_s = sz; c.z_e = ez;
    return c;
}

// lateral position of the chord where it crosses the mid plane of the major axis (extrapolated if it does not)
__device__ __forceinline__ void chord_ref(const DevCfg& g, const ChordInfo& c, float& n_ref, float& z_ref, float& sl_n, float& sl_z) {
    const int n_major = (c.cls < 2) ? g.nx : g.ny, n_minor = (c.cls < 2) ? g.ny : g.nx;
    const float m_ref = 0.5f * (float)n_major;
    const int dm = c.m_e - c.m_s;
    sl_n = 0.f; sl_z = 0.f;
    if (dm != 0) { sl_n = (float)(c.n_e - c.n_s) / (float)dm; sl_z = (float)(c.z_e - c.z_s) / (float)dm; }
    const float mid_m = 0.5f * (float)(c.m_s + c.m_e);
    n_ref = 0.5f * (float)(c.n_s + c.n_e) + sl_n * (m_ref - mid_m);
    z_ref = 0.5f * (float)(c.z_s + c.z_e) + sl_z * (m_ref - mid_m);
    n_ref = fminf(fmaxf(n_ref, -(float)n_minor), 2.f * (float)n_minor);
    z_ref = fminf(fmaxf(z_ref, 0.f), (float)(g.nz - 1));
}

__global__ void __launch_bounds__(256)
k_plan_keys(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const int32_t* __restrict__ start,
            const int32_t* __restrict__ end, int64_t m, int64_t block_size, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const uint64_t t = (uint64_t)(i / block_size);
    uint64_t key;
    if (N[i] == 0) {
        key = (t << KEY_BLOCK_SHIFT) | (7ull << (KEY_NREF_BITS + KEY_ZROW_BITS));
    } else {
        const ChordInfo c = chord_info(g, start[i], end[i]);
        float n_ref, z_ref, sl_n, sl_z;
        chord_ref(g, c, n_ref, z_ref, sl_n, sl_z);
        const int n_minor = (c.cls < 2) ? g.ny : g.nx;
        const uint64_t nq = (uint64_t)min((1 << KEY_NREF_BITS) - 1, max(0, (int)((n_ref + (float)n_minor) * 4.f)));
        const uint64_t zr = (uint64_t)min((1 << KEY_ZROW_BITS) - 1, (int)z_ref / ZROW);
        key = (t << KEY_BLOCK_SHIFT) | ((uint64_t)c.cls << (KEY_NREF_BITS + KEY_ZROW_BITS)) | (zr << KEY_NREF_BITS) | nq;
    }
    keys[i] = key;
    vals[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(256) k_plan_heads(const uint64_t* __restrict__ keys, int64_t m, uint32_t* __restrict__ head) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= m) return;
    head[j] = (j % GROUP == 0 || (keys[j] >> KEY_RUN_SHIFT) != (keys[j - 1] >> KEY_RUN_SHIFT)) ? 1u : 0u;
}

// heads write their group's start; the first head of every block writes group_begin[block]
__global__ void __launch_bounds__(256)
k_plan_starts(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ head, const uint64_t* __restrict__ gid, int64_t m,
              PlanGroup* __restrict__ groups, int64_t* __restrict__ group_begin) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= m || !head[j]) return;
    const uint64_t g = gid[j];
    groups[g].start = (uint32_t)j;
    groups[g].cls = (int)((keys[j] >> (KEY_NREF_BITS + KEY_ZROW_BITS)) & 7ull);
    const uint64_t t = keys[j] >> KEY_BLOCK_SHIFT;
    if (j == 0 || (keys[j - 1] >> KEY_BLOCK_SHIFT) != t) group_begin[t] = (int64_t)g;
}

template <typename T, typename Op>
__device__ __forceinline__ T block_reduce_256(T v, Op op, T* scratch /* 8 */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = op(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
    __syncthreads();
    T r = scratch[0];
#pragma unroll
    for (int k = 1; k < 8; ++k) r = op(r, scratch[k]);
    return r;
}

// one CTA of 256 threads per group: first row, number of slabs, window centre line
__global__ void __launch_bounds__(256)
k_plan_params(const __grid_constant__ DevCfg g, const int32_t* __restrict__ start, const int32_t* __restrict__ end,
              const uint32_t* __restrict__ perm, int64_t m, int64_t n_groups, PlanGroup* __restrict__ groups,
              uint32_t* __restrict__ cnt_len, uint32_t* __restrict__ stream_len) {
    __shared__ float sf[8];
    __shared__ int si[8];
    const int64_t gi = blockIdx.x;
    PlanGroup G = groups[gi];
    const uint32_t size = (uint32_t)(((gi + 1 < n_groups) ? (int64_t)groups[gi + 1].start : m) - (int64_t)G.start);
    if (G.cls == 7) {
        if (threadIdx.x == 0) { G.size = size; G.nslab = 0; G.m_first = 0; G.nb0 = G.zb0 = G.sn = G.sz = 0; G.wps = 0; G.cnt_off = G.stream_off = 0;
                                G.dn_lo = G.dz_lo = 0; G.dn_hi = G.dz_hi = -1; G.max_cnt = 0; groups[gi] = G; cnt_len[gi] = 0; stream_len[gi] = 0; }
        return;
    }
    const int dir = (G.cls & 1) ? -1 : 1;
    float w_sum = 0.f, wn = 0.f, wz = 0.f, wsn = 0.f, wsz = 0.f, steep = 0.f;
    int r_lo = INT_MAX, r_hi = INT_MIN;      // dir * m of starts / ends
    for (uint32_t j = threadIdx.x; j < size; j += 256) {
        const uint32_t i = perm[G.start + j];
        const ChordInfo c = chord_info(g, start[i], end[i]);
        float n_ref, z_ref, sl_n, sl_z;
        chord_ref(g, c, n_ref, z_ref, sl_n, sl_z);
        const float w = (float)abs(c.m_e - c.m_s) + 0.25f;
        w_sum += w; wn += w * n_ref; wz += w * z_ref; wsn += w * sl_n; wsz += w * sl_z;
        steep = fmaxf(steep, fabsf(sl_n) + fabsf(sl_z));              // lateral steps per row of this member's chord
        r_lo = min(r_lo, dir * c.m_s);
        r_hi = max(r_hi, dir * c.m_e);
    }
    auto fadd = [](float a, float b) { return a + b; };
    w_sum = block_reduce_256(w_sum, fadd, sf);
    wn = block_reduce_256(wn, fadd, sf);
    wz = block_reduce_256(wz, fadd, sf);
    wsn = block_reduce_256(wsn, fadd, sf);
    wsz = block_reduce_256(wsz, fadd, sf);
    steep = block_reduce_256(steep, [](float a, float b) { return fmaxf(a, b); }, sf);
    r_lo = block_reduce_256(r_lo, [](int a, int b) { return min(a, b); }, si);
    r_hi = block_reduce_256(r_hi, [](int a, int b) { return max(a, b); }, si);
    if (threadIdx.x != 0) return;
    const int n_major = (G.cls < 2) ? g.nx : g.ny;
    const float m_ref = 0.5f * (float)n_major;
    const float n_c = wn / w_sum, z_c = wz / w_sum, s_n = wsn / w_sum, s_z = wsz / w_sum;
    const int m_first = dir * r_lo;
    // centre of the tube in row r (major index m_first + dir r): n_c + s_n (m - m_ref); window = 32 (16) voxels around it
    const double n0 = (double)n_c + (double)s_n * ((double)m_first - (double)m_ref) - 0.5 * (WIN_N - 1);
    const double z0 = (double)z_c + (double)s_z * ((double)m_first - (double)m_ref) - 0.5 * (WIN_Z - 1);
    G.size = size;
    G.m_first = m_first;
    G.nslab = (r_hi - r_lo) / SLAB + 1;
    G.nb0 = (int)llrint(fmin(fmax(n0 + 0.5, -16000.0), 16000.0) * 65536.0);
    G.zb0 = (int)llrint(fmin(fmax(z0 + 0.5, -16000.0), 16000.0) * 65536.0);
    G.sn = (int)llrint((double)s_n * dir * 65536.0);
    G.sz = (int)llrint((double)s_z * dir * 65536.0);
    // words per (slab, thread) of the slab-aligned code stream, fixed BEFORE the codes are walked so that one walk can both
    // verify and emit: a member has one visit per row plus one per lateral step, i.e. 1 + |dn/dm| + |dz/dm| per row of its
    // chord, a slab SLAB rows; the steepest member's chord sets the budget, with 8 % and 3 visits of head room for
    // curvature.  A member that needs more goes to the direct list like any other that does not fit.
    const float per_slab = (float)SLAB * (1.f + fminf(steep, 2.f));
    G.wps = ((int)ceilf(per_slab * 1.08f + 3.f) + CODES_PER_WORD - 1) / CODES_PER_WORD;
    G.cnt_off = G.stream_off = 0;
    G.dn_lo = WIN_N; G.dn_hi = -1; G.dz_lo = WIN_Z; G.dz_hi = -1;      // empty; k_plan_walk widens them
    G.max_cnt = 0;
    groups[gi] = G;
    cnt_len[gi] = (uint32_t)G.nslab * GROUP;
    stream_len[gi] = (uint32_t)G.nslab * (uint32_t)G.wps * GROUP;
}

__global__ void k_plan_cnt_off(const uint64_t* __restrict__ off, int64_t n_groups, PlanGroup* __restrict__ groups) {
    const int64_t gi = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi < n_groups) groups[gi].cnt_off = off[gi];
}

// Start of k_plan_walk: thread tid of a group's CTA walks the codes of its history (plan_rank) and
// reports every visit as f(row r, code that led to it or PLAN_CODE_FIRST, in-window?) until f returns false.
struct MemberWalk {
    uint32_t pos, i, n_vis;
    int mj, n, z, r, dir, n_plus;
    const unsigned long long* cp;
};

__device__ __forceinline__ bool member_init(const DevCfg& g, const PlanGroup& G, const uint32_t* __restrict__ N,
                                            const int32_t* __restrict__ start, const uint64_t* __restrict__ code_off,
                                            const ulonglong2* __restrict__ codes, const uint32_t* __restrict__ perm, MemberWalk& mw) {
    const int rk = plan_rank((int)threadIdx.x, (int)G.size);
    if (rk < 0) return false;
    mw.pos = G.start + (uint32_t)rk;
    mw.i = perm[mw.pos];
    mw.n_vis = N[mw.i];
    const int sv = start[mw.i];
    const int vx = sv % g.nx, vy = (sv / g.nx) % g.ny;
    mw.z = sv / (g.nx * g.ny);
    mw.mj = (G.cls < 2) ? vx : vy;
    mw.n = (G.cls < 2) ? vy : vx;
    mw.dir = (G.cls & 1) ? -1 : 1;
    mw.n_plus = (G.cls < 2) ? 2 : 0;             // code of a +1 step along the minor in-plane axis
    mw.r = (mw.mj - G.m_first) * mw.dir;
    mw.cp = reinterpret_cast<const unsigned long long*>(codes + code_off[mw.i]);
    return true;
}

// One CTA per group, one thread per member: ONE walk of the member's codes that verifies the window (every visit inside
// its row's window, never a step against the travel direction, at most MAX_ROW_VISITS visits per row, at most
// 21 * wps visits per slab), records visits per slab, the packed start coordinate and the visited extent, and re-emits the
// codes slab by slab, 21 per word, words [slab][w][thread] (the stream is pre-filled with pad codes; the first visit becomes
// PLAN_CODE_FIRST).  A member that fails takes back the words it wrote and goes to its block's direct list.
__global__ void __launch_bounds__(GROUP)
k_plan_walk(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const int32_t* __restrict__ start,
            const uint64_t* __restrict__ code_off, const ulonglong2* __restrict__ codes, const uint32_t* __restrict__ perm,
            PlanGroup* __restrict__ groups, int64_t block_size, uint32_t* __restrict__ p0_out, uint8_t* __restrict__ pflag,
            uint8_t* __restrict__ cnt, unsigned long long* __restrict__ stream, uint32_t* __restrict__ direct_list,
            uint32_t* __restrict__ direct_count) {
    const PlanGroup G = groups[blockIdx.x];
    MemberWalk mw;
    if (G.cls == 7) {
        if (threadIdx.x < G.size) pflag[G.start + threadIdx.x] = 0;
        return;
    }
    if (!member_init(g, G, N, start, code_off, codes, perm, mw)) return;
    int r = mw.r, n = mw.n, z = mw.z;
    const int r_end = G.nslab * SLAB;
    bool ok = r >= 0 && r < r_end;
    uint8_t* my_cnt = cnt + G.cnt_off + threadIdx.x;
    unsigned long long* out = stream + G.stream_off + threadIdx.x;
    int cur_slab = ok ? r / SLAB : 0;
    const int first_slab = cur_slab, slab_cap = G.wps * CODES_PER_WORD;
    const uint32_t p0 = win_pack(n, r, z);
    int on_lo = WIN_N, on_hi = -1, oz_lo = WIN_Z, oz_hi = -1;
    // The loop below runs once per visit of 1.6e10 (config 2): it is written without divisions and with selects instead of
    // branches.  State: the window bases as 16.16 fixed-point accumulators (nacc = nb0 + r sn: plan_nbase without the
    // multiplication), the word being assembled (`acc`: every code enters at the top and moves down 3 bits per push, so no
    // variable shift per visit), kw = codes in it, k = codes in the slab, op = where the next word of the slab goes.
    long long nacc = (long long)G.nb0 + (long long)r * G.sn, zacc = (long long)G.zb0 + (long long)r * G.sz;
    unsigned long long w = 0, acc = ~0ull;
    unsigned long long* op = out + (size_t)cur_slab * G.wps * GROUP;
    int nrem = 0, row_cnt = 0, k = 0, kw = 0;
    // codes sit at the top 3 kw bits of acc, oldest lowest: move them down, pads (all ones) above; bit 63 of a full word is a pad bit
    auto finish_word = [&]() -> unsigned long long {
        return kw == CODES_PER_WORD ? ((acc >> 1) | 0x8000000000000000ull) : ((acc >> (64 - 3 * kw)) | (~0ull << (3 * kw)));
    };
    const int cls = G.cls;
    // one exit test per visit: a failed check sets `bad`, the visit is not emitted, and the loop condition ends the walk
    bool bad = !ok;
    for (uint32_t v = 0; v < mw.n_vis && !bad; ++v) {
        int code = PLAN_CODE_FIRST;
        if (v > 0) {
            if (nrem == 0) { w = __ldg(mw.cp++); nrem = CODES_PER_WORD; }
            code = (int)((unsigned)w & 7u);
            w >>= 3; --nrem;
            const bool is_row = code == cls;
            bad = (code == (cls ^ 1)) | (code >= 6);                                  // against the travel direction, or not a step
            const int sign = 1 - 2 * (code & 1);                                      // even code = +1 along its axis
            const bool is_z = code >= 4;
            z += is_z ? sign : 0;
            n += (is_z | is_row) ? 0 : sign;
            r += is_row ? 1 : 0;
            nacc += is_row ? (long long)G.sn : 0ll;
            zacc += is_row ? (long long)G.sz : 0ll;
            row_cnt = is_row ? 0 : row_cnt;
            if (is_row && (r & (SLAB - 1)) == 0) {                                    // first row of the next slab
                if (r >= r_end) bad = true;
                else {
                    if (kw != 0) *op = finish_word();
                    my_cnt[(size_t)cur_slab * GROUP] = (uint8_t)k;
                    ++cur_slab; k = 0; kw = 0; acc = ~0ull;
                    op = out + (size_t)cur_slab * G.wps * GROUP;
                }
            }
        }
        const int dn = n - (int)(nacc >> 16), dz = z - (int)(zacc >> 16);
        bad |= ((unsigned)dn >= (unsigned)WIN_N) | ((unsigned)dz >= (unsigned)WIN_Z) | (++row_cnt > MAX_ROW_VISITS) | (k >= slab_cap);
        if (!bad) {
            on_lo = min(on_lo, dn); on_hi = max(on_hi, dn); oz_lo = min(oz_lo, dz); oz_hi = max(oz_hi, dz);
            acc = (acc >> 3) | ((unsigned long long)(unsigned)code << 61);
            ++k;
            if (++kw == CODES_PER_WORD) { *op = (acc >> 1) | 0x8000000000000000ull; op += GROUP; kw = 0; acc = ~0ull; }
        }
    }
    ok = !bad;
    if (ok) {
        if (kw != 0) *op = finish_word();
        my_cnt[(size_t)cur_slab * GROUP] = (uint8_t)k;
        // widen the group's visited extent (the plain read only filters out the atomics that cannot change anything)
        PlanGroup* Gp = groups + blockIdx.x;
        if (on_lo < *(volatile int32_t*)&Gp->dn_lo) atomicMin(&Gp->dn_lo, on_lo);
        if (on_hi > *(volatile int32_t*)&Gp->dn_hi) atomicMax(&Gp->dn_hi, on_hi);
        if (oz_lo < *(volatile int32_t*)&Gp->dz_lo) atomicMin(&Gp->dz_lo, oz_lo);
        if (oz_hi > *(volatile int32_t*)&Gp->dz_hi) atomicMax(&Gp->dz_hi, oz_hi);
        p0_out[mw.pos] = p0;
        pflag[mw.pos] = 1;
    } else {
        // take back what was written: the thread's words of the slabs it reached are pads again, its counts zero
        const int last = min(cur_slab, G.nslab - 1);
        for (int s = max(first_slab, 0); s <= last; ++s) {
            for (int wi = 0; wi < G.wps; ++wi) out[((size_t)s * G.wps + wi) * GROUP] = ~0ull;
            my_cnt[(size_t)s * GROUP] = 0;
        }
        pflag[mw.pos] = 0;
        const uint64_t t = (uint64_t)mw.i / (uint64_t)block_size;
        const uint32_t slot = atomicAdd(direct_count + t, 1u);
        direct_list[t * (uint64_t)block_size + slot] = mw.i;
    }
}

__global__ void k_plan_stream_off(const uint64_t* __restrict__ off, int64_t n_groups, PlanGroup* __restrict__ groups) {
    const int64_t gi = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi < n_groups) groups[gi].stream_off = off[gi];
}

// launch order of a block's groups: key = (block, -work), work = slabs x words per slab x members
__global__ void k_plan_work_keys(const PlanGroup* __restrict__ groups, const uint32_t* __restrict__ perm, int64_t n_groups,
                                 int64_t block_size, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    const int64_t gi = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi >= n_groups) return;
    const PlanGroup G = groups[gi];
    const uint64_t t = (uint64_t)perm[G.start] / (uint64_t)block_size;
    const uint32_t work = (uint32_t)G.nslab * (uint32_t)G.wps * G.size;
    keys[gi] = (t << 32) | (uint64_t)(0xffffffffu - work);
    vals[gi] = (uint32_t)gi;
}

// totals of one sweep for pct_plan_info: window slots staged (= the visited extent of every slab row that lies inside the
// grid; an upper bound of the flushed slots), windowed histories and their visits.  tot = {slots, histories, visits}.
__global__ void __launch_bounds__(256)
k_plan_totals(const __grid_constant__ DevCfg g, const PlanGroup* __restrict__ groups, int64_t n_groups, const uint32_t* __restrict__ perm,
              const uint8_t* __restrict__ pflag, const uint32_t* __restrict__ N, int64_t m, unsigned long long* __restrict__ tot) {
    __shared__ unsigned long long sh[3][8];
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, span = m > n_groups ? m : n_groups;
    unsigned long long slots = 0, hist = 0, vis = 0;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < span; j += stride) {
        if (j < n_groups) {
            const PlanGroup G = groups[j];
            if (G.cls != 7 && G.wps > 0 && G.dn_hi >= G.dn_lo && G.dz_hi >= G.dz_lo) {
                const int dim_m = G.cls < 2 ? g.nx : g.ny, dir = (G.cls & 1) ? -1 : 1;
                int rows = 0;
                for (int r = 0; r < G.nslab * SLAB; ++r) rows += (unsigned)(G.m_first + dir * r) < (unsigned)dim_m;
                slots += (unsigned long long)rows * (unsigned)(G.dn_hi - G.dn_lo + 1) * (unsigned)(G.dz_hi - G.dz_lo + 1);
            }
        }
        if (j < m && pflag[j]) { ++hist; vis += N[perm[j]]; }
    }
    // one atomic per CTA and counter (same-address atomics serialise in L2)
    unsigned long long v[3] = {slots, hist, vis};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
        if ((threadIdx.x & 31) == 0) sh[k][threadIdx.x >> 5] = v[k];
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        unsigned long long a = 0;
        for (int w = 0; w < 8; ++w) a += sh[threadIdx.x][w];
        if (a) atomicAdd(tot + threadIdx.x, a);
    }
}

void free_solve_plan(SolvePlan* plan) {
    if (!plan) return;
    cudaDeviceSynchronize();         // freed on the legacy stream: nothing may still use the plan
    cache_free(plan->perm); cache_free(plan->p0); cache_free(plan->pflag); cache_free(plan->cnt); cache_free(plan->groups); cache_free(plan->stream); cache_free(plan->launch_order);
    cache_free(plan->direct_list); cache_free(plan->d_direct_count);
    delete plan;
}

int build_solve_plan(pct_ctx* ctx, const pct_paths* P, int64_t block_size, cudaStream_t st, SolvePlan** out) {
    *out = nullptr;
    const int64_t m = P->m;
    const int64_t n_blocks = (m + block_size - 1) / block_size;
    if (m <= 0 || m >= 0xffffffffLL || n_blocks >= (1LL << 24)) return set_error(ctx, PCT_E_INVALID_ARG, "solve plan: size out of range");
    SolvePlan* plan = new (std::nothrow) SolvePlan();
    if (!plan) return set_error(ctx, PCT_E_OOM, "host allocation");
    plan->block_size = block_size; plan->n_blocks = n_blocks; plan->n_groups = 0; plan->n_direct = 0; plan->cnt_bytes = 0;
    plan->staged_slots = plan->windowed_histories = plan->windowed_visits = 0;
    plan->perm = nullptr; plan->p0 = nullptr; plan->pflag = nullptr; plan->cnt = nullptr; plan->groups = nullptr;
    plan->direct_list = nullptr; plan->d_direct_count = nullptr; plan->stream = nullptr; plan->stream_words = 0; plan->launch_order = nullptr;
    uint64_t *keysA = nullptr, *keysB = nullptr, *cnt_off = nullptr;
    uint32_t *valsA = nullptr, *valsB = nullptr, *cnt_len = nullptr, *stream_len = nullptr;
    void* tmp = nullptr;
    int64_t* d_group_begin = nullptr;
    auto fail = [&](int code) {
        cache_free(keysA); cache_free(keysB); cache_free(valsA); cache_free(valsB); cache_free(tmp); cache_free(cnt_off); cache_free(cnt_len); cache_free(stream_len);
        cache_free(d_group_begin);
        free_solve_plan(plan);
        return code;
    };
#define PLAN_CUDA(call)                                                                                         \
    do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError();                               \
        return fail(set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
    const size_t mm = (size_t)m;
    const bool dbg = getenv("PCT_PLAN_DEBUG") != nullptr;
    auto t_last = std::chrono::steady_clock::now();
    auto lap = [&](const char* what) {
        if (!dbg) return;
        cudaStreamSynchronize(st);
        const auto now = std::chrono::steady_clock::now();
        unsigned long long reserved = 0, used = 0, thr = 0;
        cudaMemPool_t pool;
        if (cudaDeviceGetMemPool(&pool, ctx->device) == cudaSuccess) {
            cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReservedMemCurrent, &reserved);
            cudaMemPoolGetAttribute(pool, cudaMemPoolAttrUsedMemCurrent, &used);
            cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        }
        fprintf(stderr, "[plan] %-28s %8.2f ms   pool reserved %.2f GB used %.2f GB thr %.3g\n", what,
                std::chrono::duration<double, std::milli>(now - t_last).count(), reserved / 1e9, used / 1e9, (double)thr);
        t_last = now;
    };
    PLAN_CUDA(cache_alloc((void**)&keysA, 8 * mm)); PLAN_CUDA(cache_alloc((void**)&keysB, 8 * mm));
    PLAN_CUDA(cache_alloc((void**)&valsA, 4 * mm)); PLAN_CUDA(cache_alloc((void**)&valsB, 4 * mm));
    const unsigned nb256 = (unsigned)((m + 255) / 256);
    k_plan_keys<<<nb256, 256, 0, st>>>(ctx->cfg, P->N, P->start, P->end, m, block_size, keysA, valsA);
    ++ctx->launches;
    PLAN_CUDA(cudaGetLastError());
    int block_bits = 1;
    while ((1LL << block_bits) < n_blocks) ++block_bits;
    cub::DoubleBuffer<uint64_t> dk(keysA, keysB);
    cub::DoubleBuffer<uint32_t> dv(valsA, valsB);
    size_t tmp_bytes = 0;
    PLAN_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, dk, dv, m, 0, KEY_BLOCK_SHIFT + block_bits, st));
    PLAN_CUDA(cache_alloc((void**)&tmp, tmp_bytes > 0 ? tmp_bytes : 16));
    PLAN_CUDA(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, dk, dv, m, 0, KEY_BLOCK_SHIFT + block_bits, st));
    const uint64_t* keys = dk.Current();
    uint64_t* gid = dk.Alternate();            // reused: group id per sorted position
    uint32_t* head = dv.Alternate();           // reused: head flags
    plan->perm = dv.Current();
    if (plan->perm == valsA) valsA = nullptr; else valsB = nullptr;   // ownership moved to the plan
    lap("keys + sort");
    k_plan_heads<<<nb256, 256, 0, st>>>(keys, m, head);
    ++ctx->launches;
    PLAN_CUDA(cudaGetLastError());
    int rc;
    if ((rc = launch_scan_u32(ctx, head, gid, m, 0, ctx->d_total, st)) != PCT_OK) return fail(rc);
    unsigned long long n_groups = 0;
    PLAN_CUDA(cudaMemcpyAsync(&n_groups, ctx->d_total, sizeof(n_groups), cudaMemcpyDeviceToHost, st));
    PLAN_CUDA(cudaStreamSynchronize(st));
    plan->n_groups = (int64_t)n_groups;
    PLAN_CUDA(cache_alloc((void**)&plan->groups, sizeof(PlanGroup) * (size_t)(n_groups + 1)));
    PLAN_CUDA(cache_alloc((void**)&d_group_begin, sizeof(int64_t) * (size_t)(n_blocks + 1)));
    PLAN_CUDA(cache_alloc((void**)&cnt_len, sizeof(uint32_t) * (size_t)n_groups));
    PLAN_CUDA(cache_alloc((void**)&stream_len, sizeof(uint32_t) * (size_t)n_groups));
    PLAN_CUDA(cache_alloc((void**)&cnt_off, sizeof(uint64_t) * (size_t)n_groups));
    lap("heads + scan");
    k_plan_starts<<<nb256, 256, 0, st>>>(keys, head, gid, m, plan->groups, d_group_begin);
    k_plan_params<<<(unsigned)n_groups, 256, 0, st>>>(ctx->cfg, P->start, P->end, plan->perm, m, (int64_t)n_groups, plan->groups, cnt_len, stream_len);
    ctx->launches += 2;
    PLAN_CUDA(cudaGetLastError());
    // offsets of every group's visit-count table and of its slab-aligned code stream: both sizes are known before the walk
    unsigned long long cnt_bytes = 0, stream_words = 0;
    if ((rc = launch_scan_u32(ctx, cnt_len, cnt_off, (int64_t)n_groups, 0, ctx->d_total, st)) != PCT_OK) return fail(rc);
    PLAN_CUDA(cudaMemcpyAsync(&cnt_bytes, ctx->d_total, sizeof(cnt_bytes), cudaMemcpyDeviceToHost, st));
    k_plan_cnt_off<<<(unsigned)((n_groups + 255) / 256), 256, 0, st>>>(cnt_off, (int64_t)n_groups, plan->groups);
    PLAN_CUDA(cudaStreamSynchronize(st));
    if ((rc = launch_scan_u32(ctx, stream_len, cnt_off, (int64_t)n_groups, 0, ctx->d_total, st)) != PCT_OK) return fail(rc);
    PLAN_CUDA(cudaMemcpyAsync(&stream_words, ctx->d_total, sizeof(stream_words), cudaMemcpyDeviceToHost, st));
    k_plan_stream_off<<<(unsigned)((n_groups + 255) / 256), 256, 0, st>>>(cnt_off, (int64_t)n_groups, plan->groups);
    ctx->launches += 2;
    // the sort buffers are no longer needed once the group table is complete
    PLAN_CUDA(cudaStreamSynchronize(st));
    plan->cnt_bytes = (int64_t)cnt_bytes;
    plan->stream_words = (int64_t)stream_words;
    cache_free(keysA); cache_free(keysB); cache_free(valsA); cache_free(valsB); cache_free(tmp);
    keysA = keysB = nullptr; valsA = valsB = nullptr; tmp = nullptr;
    lap("starts + params + scans");
    PLAN_CUDA(cache_alloc((void**)&plan->cnt, cnt_bytes > 0 ? (size_t)cnt_bytes : 16));
    PLAN_CUDA(cudaMemsetAsync(plan->cnt, 0, cnt_bytes > 0 ? (size_t)cnt_bytes : 16, st));
    PLAN_CUDA(cache_alloc((void**)&plan->stream, stream_words > 0 ? 8 * (size_t)stream_words : 16));
    PLAN_CUDA(cudaMemsetAsync(plan->stream, 0xFF, stream_words > 0 ? 8 * (size_t)stream_words : 16, st));
    PLAN_CUDA(cache_alloc((void**)&plan->p0, 4 * mm));
    PLAN_CUDA(cache_alloc((void**)&plan->pflag, mm));
    PLAN_CUDA(cache_alloc((void**)&plan->direct_list, 4 * mm));
    PLAN_CUDA(cache_alloc((void**)&plan->d_direct_count, sizeof(uint32_t) * (size_t)n_blocks));
    PLAN_CUDA(cudaMemsetAsync(plan->d_direct_count, 0, sizeof(uint32_t) * (size_t)n_blocks, st));
    lap("allocs + memsets");
    k_plan_walk<<<(unsigned)n_groups, GROUP, 0, st>>>(ctx->cfg, P->N, P->start, P->code_off, P->codes, plan->perm, plan->groups, block_size,
                                                     plan->p0, plan->pflag, plan->cnt, plan->stream, plan->direct_list, plan->d_direct_count);
    ++ctx->launches;
    PLAN_CUDA(cudaGetLastError());
    lap("walk (verify + emit)");
    {   // longest-first launch order inside every block
        uint64_t *wk0 = nullptr, *wk1 = nullptr;
        uint32_t *wv0 = nullptr, *wv1 = nullptr;
        void* wtmp = nullptr;
        const size_t ng = (size_t)n_groups;
        auto wfree = [&]() { cache_free(wk0); cache_free(wk1); cache_free(wv0); cache_free(wv1); cache_free(wtmp); };
#define WORK_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError(); wfree(); \
        return fail(set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
        WORK_CUDA(cache_alloc((void**)&wk0, 8 * ng)); WORK_CUDA(cache_alloc((void**)&wk1, 8 * ng));
        WORK_CUDA(cache_alloc((void**)&wv0, 4 * ng)); WORK_CUDA(cache_alloc((void**)&wv1, 4 * ng));
        k_plan_work_keys<<<(unsigned)((n_groups + 255) / 256), 256, 0, st>>>(plan->groups, plan->perm, (int64_t)n_groups, block_size, wk0, wv0);
        cub::DoubleBuffer<uint64_t> wk(wk0, wk1);
        cub::DoubleBuffer<uint32_t> wv(wv0, wv1);
        size_t wbytes = 0;
        WORK_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, wbytes, wk, wv, (int64_t)n_groups, 0, 32 + block_bits, st));
        WORK_CUDA(cache_alloc((void**)&wtmp, wbytes > 0 ? wbytes : 16));
        WORK_CUDA(cub::DeviceRadixSort::SortPairs(wtmp, wbytes, wk, wv, (int64_t)n_groups, 0, 32 + block_bits, st));
        WORK_CUDA(cudaStreamSynchronize(st));
        plan->launch_order = wv.Current();
        if (plan->launch_order == wv0) wv0 = nullptr; else wv1 = nullptr;
        wfree();
#undef WORK_CUDA
        ++ctx->launches;
    }
    lap("launch order");
    {   // per-sweep totals for the roofline report
        unsigned long long* d_tot = nullptr;
        unsigned long long h_tot[3] = {0, 0, 0};
        PLAN_CUDA(cache_alloc((void**)&d_tot, sizeof(h_tot)));
        cudaError_t e = cudaMemsetAsync(d_tot, 0, sizeof(h_tot), st);
        if (e == cudaSuccess) {
            k_plan_totals<<<(unsigned)(ctx->num_sms * 8), 256, 0, st>>>(ctx->cfg, plan->groups, (int64_t)n_groups, plan->perm, plan->pflag, P->N, m, d_tot);
            ++ctx->launches;
            e = cudaMemcpyAsync(h_tot, d_tot, sizeof(h_tot), cudaMemcpyDeviceToHost, st);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cache_free(d_tot);
        PLAN_CUDA(e);
        plan->staged_slots = (int64_t)h_tot[0]; plan->windowed_histories = (int64_t)h_tot[1]; plan->windowed_visits = (int64_t)h_tot[2];
    }
    plan->counts_ready.assign((size_t)n_blocks, 0);      // the count cache itself belongs to the context (pct_solve)
    plan->group_begin.resize((size_t)n_blocks + 1);
    plan->direct_count.resize((size_t)n_blocks);
    PLAN_CUDA(cudaMemcpyAsync(plan->group_begin.data(), d_group_begin, sizeof(int64_t) * (size_t)n_blocks, cudaMemcpyDeviceToHost, st));
    PLAN_CUDA(cudaMemcpyAsync(plan->direct_count.data(), plan->d_direct_count, sizeof(uint32_t) * (size_t)n_blocks, cudaMemcpyDeviceToHost, st));
    PLAN_CUDA(cudaStreamSynchronize(st));
    plan->group_begin[(size_t)n_blocks] = (int64_t)n_groups;
    for (uint32_t c : plan->direct_count) plan->n_direct += c;
    cache_free(cnt_off); cache_free(cnt_len); cache_free(stream_len); cache_free(d_group_begin);
#undef PLAN_CUDA
    *out = plan;
    return PCT_OK;
}

}  // namespace pct
