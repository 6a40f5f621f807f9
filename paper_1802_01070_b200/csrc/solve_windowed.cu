// solve_windowed.cu -- K2w: the block projection (A4-A6: gather a_i.x, residual, scatter {c_i, 1}, R14-R17)
// for the histories a solve plan has verified to stay inside their group's window (plan.cu, DESIGN.md 5.3/5.4).
//
// One CTA per group, one thread per history.  The CTA marches along the group's major axis in slabs of SLAB rows; the
// window of a slab (WIN_N x SLAB x WIN_Z voxels) lives in shared memory:
//   pass 1  the slab's x values are staged with coalesced loads, every thread walks the part of its row that lies in
//           the slab (3-bit code -> table {delta, field mask} -> packed circular coordinate -> LDS) and adds up S_i;
//   then    c_i = (b_i - l_i S_i) / (N_i l_i)  (R17), CTA-wide max |c_i| -> power-of-two fixed-point scale (R21);
//   pass 2  the same walk adds round(c_i 2^e) and 1 to the slab's {Delta, s} window with native 32-bit shared-memory
//           atomics (ATOMS.ADD), the CTA flushes the touched slots to the global accumulator with coalesced
//           red.global.add.v2.f32 and clears them.
// x is frozen during a block (R14): it is only read.  Global reductions drop from one per visit to one per touched
// voxel per group and slab; gathers never leave the SM.
#include "pct_internal.cuh"

namespace pct {

// pass 1: two float x[8192] buffers; pass 2: int Delta[8192], uint s[8192] (or a second Delta copy).  The 64 KB window is
// aligned to 32 KB inside the allocation so that a thread's packed coordinate can carry the window's shared address in
// its upper bits (field arithmetic touches bits 2-14 only): no base addition per visit.
constexpr int K2W_WIN = WIN_SLOTS * 8;
constexpr int K2W_SMEM = K2W_WIN + 32768;
// Fixed-point Delta (R21): |c_i| 2^e < 2^FIX and at most A additions per slot must satisfy A 2^FIX < 2^31.  The counting
// sweep only knows A <= MAX_ROW_VISITS * GROUP = 6144 (FIX = 17) and measures the true maximum; later sweeps use it.
constexpr int FIX_BITS = 17;

__device__ __forceinline__ void red_add_v2_w(float2* p, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

struct WinGeom {
    int dir, stride_m, stride_n, stride_z, dim_m, dim_n, dim_z;
    bool x_major;
};

// Staging and flushing: thread tid owns the window column (nq, ml) = f(tid) and the STAGE_Z slots zq = zq0 + 2k of
// it.  The lane index runs along the grid's x axis (the contiguous one): the minor axis for y-major groups, the row
// (major) axis for x-major groups, so that global loads and reductions coalesce.
constexpr int STAGE_Z = WIN_SLOTS / GROUP;   // 8

struct Column {
    int base;        // voxel index of (row, n, z = 0), or -1 if the column lies outside the grid in n or in the row
    int zb;          // first slice of the window in this row
    int on;          // n offset of the column from the row's window base
};

// Calls f(z, byte offset of the slot) for the slots of a thread's column that the group's members can visit
// (PlanGroup::dn_*, dz_*) and that lie inside the grid.  The thread owns the slots of one parity of z; col_a0 = window
// offset of the column for z = 0 (the swizzle only involves the parity of z, a thread constant).
template <typename F>
__device__ __forceinline__ void for_visited_slots(const PlanGroup& G, const Column& col, int zq0, unsigned col_a0, int dim_z, F&& f) {
    if (col.base < 0 || col.on < G.dn_lo || col.on > G.dn_hi) return;
    const int o0 = (zq0 - col.zb) & 1;                                   // this thread's offsets from zb: o0, o0 + 2, ...
    const int lo = max(G.dz_lo, -col.zb), hi = min(G.dz_hi, dim_z - 1 - col.zb);
    const int k_hi = min(STAGE_Z - 1, (hi - o0) >> 1);
    for (int k = max(0, (lo - o0 + 1) >> 1); k <= k_hi; ++k) {
        const int z = col.zb + o0 + 2 * k;
        f(z, col_a0 + ((unsigned)(z & (WIN_Z - 1)) << 11));
    }
}

__device__ __forceinline__ Column slab_column(const PlanGroup& G, const WinGeom& w, int s, int nq, int ml) {
    const int r = s * SLAB + ml;
    const int nb = plan_nbase(G, r);
    Column c;
    c.on = (nq - nb) & (WIN_N - 1);
    const int n = nb + c.on;
    const int mj = G.m_first + w.dir * r;
    c.zb = plan_zbase(G, r);
    c.base = ((unsigned)n < (unsigned)w.dim_n && (unsigned)mj < (unsigned)w.dim_m) ? mj * w.stride_m + n * w.stride_n : -1;
    return c;
}

__device__ __forceinline__ float lds_f32(unsigned a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ unsigned lds_u32(unsigned a) { unsigned v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void red_add_f32(float* p, float a) { asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(a) : "memory"); }
__device__ __forceinline__ void atoms_add(unsigned a, int v) { asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
// 4-byte asynchronous global -> shared copy; valid == false writes a zero instead (src-size 0)
__device__ __forceinline__ void cp_async_f32(unsigned dst, const float* src, bool valid) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(valid ? 4 : 0) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void atoms_inc(unsigned a) { asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(a) : "memory"); }

// One slab of one thread's walk.  The slab's codes sit in G.wps words [slab][w][thread] (21 codes each, pad = 7); the
// loop runs to the warp's largest visit count (rounded up to 3) so that all lanes stay converged.  visit(p) is called
// on every real visit.  tbl_s = shared address of the step table; entry = delta | field mask << 16; 0 marks a pad.
// w0 = the slab's first word (loaded by the caller ahead of time).
template <typename F>
__device__ __forceinline__ void walk_slab(const unsigned long long* __restrict__ sp, unsigned long long w0, int cmax,
                                          unsigned tbl_s, unsigned& p, F&& visit) {
    for (int wi = 0; wi * CODES_PER_WORD < cmax; ++wi) {
        const unsigned long long w = wi == 0 ? w0 : __ldg(sp + (size_t)wi * GROUP);
        const int lim = cmax - wi * CODES_PER_WORD;          // warp-uniform
#pragma unroll
        for (int k3 = 0; k3 < CODES_PER_WORD; k3 += 3) {
            if (k3 >= lim) break;
#pragma unroll
            for (int k = k3; k < k3 + 3; ++k) {
                const unsigned code4 = (unsigned)(w >> (3 * k)) << 2 & 0x1Cu;
                const unsigned t = lds_u32(tbl_s + code4);              // delta | mask << 16; 0 = pad
                const unsigned fm = t >> 16;
                p = ((p + t) & fm) | (p & ~fm);                        // the mask half of t is discarded by the select
                if (t != 0u) visit(p);
            }
        }
    }
}

// One history's row walked with red.global.add.f32 of `c` on every visit (the "late" members of k_block_windowed: outliers
// and non-finite residuals, R21).  acc[v * stride] is the Delta accumulator of voxel v.
__device__ __noinline__ void late_walk(int sx, int sy, int sz, const ulonglong2* __restrict__ codes, uint64_t off, int32_t v, uint32_t n_vis,
                                       float c, float* __restrict__ acc, int stride) {
    const unsigned long long* cp = reinterpret_cast<const unsigned long long*>(codes + off);
    unsigned long long w = 0ull;
    for (uint32_t k = 0; k < n_vis; ++k) {
        if (k > 0) {
            const uint32_t f = (k - 1) % CODES_PER_WORD;
            if (f == 0) w = __ldg(cp++);
            const int code = (int)((w >> (3 * f)) & 7ull);
            const int mag = (code >> 1) == 0 ? sx : ((code >> 1) == 1 ? sy : sz);
            v += (code & 1) ? -mag : mag;
        }
        red_add_f32(acc + (size_t)v * stride, c);
    }
}

// Median binade of the finite |c_i| of a CTA from the exponent histogram (256 bins); -1 if there is none.  One warp.
__device__ __noinline__ int median_binade(const unsigned* ehist, int lane) {
    unsigned mine = 0u;
#pragma unroll
    for (int k = 0; k < 8; ++k) mine += ehist[lane * 8 + k];
    unsigned incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
    const unsigned total = __shfl_sync(0xffffffffu, incl, 31), half = (total + 1u) >> 1;
    const unsigned at = __ballot_sync(0xffffffffu, incl >= half && total > 0u);
    int bin = -1;
    if (total > 0u && lane == __ffs(at) - 1) {
        unsigned cum = incl - mine;
        bin = lane * 8;
        for (int k = 0; k < 8; ++k) { cum += ehist[lane * 8 + k]; if (cum >= half) { bin = lane * 8 + k; break; } }
    }
    return __reduce_max_sync(0xffffffffu, bin);
}

// COUNT = true: fused column counts, {Delta_j, s_j} go to the float2 accumulator `ds` (first sweep over a block, or no
// count cache).  COUNT = false: s_j^t is already cached per block (it does not depend on x, R15), only Delta_j is
// accumulated, into `dsum`; the freed half of the window holds a second copy of Delta (odd / even lanes) to halve the
// serialisation of same-address shared atomics.
template <bool COUNT>
__global__ void __launch_bounds__(GROUP, 2)
k_block_windowed(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const float* __restrict__ ell,
                 const int32_t* __restrict__ start, const uint64_t* __restrict__ code_off, const ulonglong2* __restrict__ codes,
                 const uint32_t* __restrict__ perm, const uint32_t* __restrict__ p0, const uint8_t* __restrict__ pflag,
                 const uint8_t* __restrict__ cnt, const unsigned long long* __restrict__ stream,
                 PlanGroup* __restrict__ groups, const uint32_t* __restrict__ launch_order, int64_t group0, const float* __restrict__ b,
                 const float* __restrict__ wts, const float* __restrict__ x,
                 float2* __restrict__ ds, float* __restrict__ dsum) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ unsigned tbl[8];
    __shared__ float red[GROUP / 32];
    __shared__ unsigned ehist[256];               // members per binade of |c_i| (R21: robust fixed-point scale)
    __shared__ int e_med;
    __shared__ PlanGroup Gs;
    if (threadIdx.x == 0) Gs = groups[launch_order[group0 + blockIdx.x]];
    if (threadIdx.x < 256) ehist[threadIdx.x] = 0u;
    __syncthreads();
    const PlanGroup& G = Gs;
    if (G.cls == 7 || G.nslab == 0 || G.wps == 0) return;
    const int tid = threadIdx.x;
    WinGeom wg;
    wg.x_major = G.cls < 2;
    wg.dir = (G.cls & 1) ? -1 : 1;
    wg.stride_m = wg.x_major ? 1 : g.nx; wg.stride_n = wg.x_major ? g.nx : 1; wg.stride_z = g.nx * g.ny;
    wg.dim_m = wg.x_major ? g.nx : g.ny; wg.dim_n = wg.x_major ? g.ny : g.nx; wg.dim_z = g.nz;
    if (tid < 8) {
        // {delta, field mask} of a step: fields are n (bits 2-6), row (7-10), z (11-14); additions wrap inside a field.
        // PLAN_CODE_FIRST (6) and pad (7) do not move; the pad's entry is 0.
        const int n_plus = wg.x_major ? 2 : 0;
        unsigned e = tid == PLAN_CODE_FIRST ? 0x80000000u : 0u;     // mask bit 15 of p: never set, so no move
        if (tid == G.cls) e = 0x80u | 0x780u << 16;
        else if (tid == n_plus) e = 0x4u | 0x7Cu << 16;
        else if (tid == n_plus + 1) e = 0x7Cu | 0x7Cu << 16;
        else if (tid == 4) e = 0x800u | 0x7800u << 16;
        else if (tid == 5) e = 0x7800u | 0x7800u << 16;
        tbl[tid] = e;
    }
    const int rk = plan_rank(tid, (int)G.size);
    const bool active = rk >= 0 && pflag[G.start + rk] != 0;
    uint32_t i = 0, n_vis = 0;
    unsigned p_init = 0;
    if (active) {
        i = perm[G.start + rk];
        n_vis = N[i];
        p_init = p0[G.start + rk];
    }
    const unsigned raw_s = (unsigned)__cvta_generic_to_shared(smem), tbl_s = (unsigned)__cvta_generic_to_shared(tbl);
    const unsigned win_s = (raw_s + 0x7FFFu) & ~0x7FFFu;                      // 32 KB aligned
    unsigned char* const win = smem + (win_s - raw_s);
    const uint8_t* my_cnt = cnt + G.cnt_off + tid;
    const unsigned long long* my_stream = stream + G.stream_off + tid;
    // this thread's window column for staging / flushing
    const int col_nq = wg.x_major ? (tid >> 4) & (WIN_N - 1) : tid & (WIN_N - 1);
    const int col_ml = wg.x_major ? tid & (SLAB - 1) : (tid >> 5) & (SLAB - 1);
    const int col_zq0 = tid >> 9;                                            // 0 or 1; slots zq0 + 2k
    const unsigned col_a0 = win_addr(win_pack(col_nq, col_ml, col_zq0)) - ((unsigned)col_zq0 << 11);   // the column's slot for z = 0

    // ---- pass 1: S_i = sum of x over the visits ----------------------------------------------------------------------
    // The x window is double buffered in the two halves of the shared window (pass 1 needs 32 KB of the 64 KB): slab
    // s + 1 is staged with cp.async while slab s is walked, one barrier per slab.
    auto stage = [&](int s) {
        const Column col = slab_column(G, wg, s, col_nq, col_ml);
        const unsigned dst = win_s + (unsigned)(s & 1) * (WIN_SLOTS * 4);
        for_visited_slots(G, col, col_zq0, col_a0, wg.dim_z, [&](int z, unsigned off) {
            cp_async_f32(dst + off, x + (col.base + z * wg.stride_z), true);
        });
    };
    unsigned p = win_s + p_init;                  // window address + packed coordinate; starts in x buffer 0
    float S = 0.f;
    stage(0);
    unsigned long long w_next = __ldg(my_stream);
    int c_next = (int)__ldg(my_cnt);              // visits in the slab; 0 for threads without a (windowed) history
    for (int s = 0; s < G.nslab; ++s) {
        const int c = c_next;
        const unsigned long long w0 = w_next;
        cp_async_wait_all();
        __syncthreads();                          // slab s is staged; slab s - 1 is walked (and tbl is visible)
        if (s + 1 < G.nslab) {                    // the next slab's x window, first word and count are on their way during the walk
            stage(s + 1);
            w_next = __ldg(my_stream + (size_t)(s + 1) * G.wps * GROUP);
            c_next = (int)__ldg(my_cnt + (size_t)(s + 1) * GROUP);
        }
        const int cmax = __reduce_max_sync(0xffffffffu, c);
        if (s > 0) p += (s & 1) ? 0x8000u : 0xFFFF8000u;          // switch to the other x buffer (the fields sit below bit 15)
        walk_slab(my_stream + (size_t)s * G.wps * GROUP, w0, cmax, tbl_s, p, [&](unsigned q) { S += lds_f32(win_addr(q)); });
    }
    // ---- c_i and the CTA's fixed-point scale (R17, R21) -----------------------------------------------------------------
    // The scale must not be set by an outlier (an absurd WEPL makes |c_i| orders of magnitude larger than its neighbours'
    // and would coarsen the quantum of all 1024 members) nor by a non-finite value.  So: the CTA takes the MEDIAN binade
    // of the finite |c_i| (histogram of the FP32 exponents), caps the scale at 512 x that binade, and every member whose
    // c_i is not finite or lies beyond the cap is "late": it adds nothing to the fixed-point window and instead walks its
    // row once with red.global.add.f32, exactly as the direct kernel does (Inf / NaN propagate the same way).
    float ci = 0.f;
    const bool has = active && n_vis > 0;
    if (has) {
        const float l = ell[i];
        ci = (b[i] - l * S) / ((float)n_vis * l);
        if (wts) ci *= wts[i];                                   // R27: weighted row
    }
    const float aci = fabsf(ci);
    const bool finite = aci < INFINITY;                                  // false for Inf and NaN
    {
        const unsigned e = (has && finite && aci > 0.f) ? (__float_as_uint(aci) >> 23) : 0xFFFFFFFFu;
        const unsigned peers = __match_any_sync(0xffffffffu, e);
        if (e != 0xFFFFFFFFu && (tid & 31) == __ffs(peers) - 1) atomicAdd(&ehist[e], (unsigned)__popc(peers));
    }
    float mx = finite ? aci : 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    __syncthreads();                              // all walkers done with xs; ehist complete
    if ((tid & 31) == 0) red[tid >> 5] = mx;
    int* dl = reinterpret_cast<int*>(win);
#pragma unroll
    for (int k = 0; k < 2 * WIN_SLOTS / GROUP; ++k) dl[tid + k * GROUP] = 0;      // clears Delta and s
    if (tid < 32) { const int m = median_binade(ehist, tid); if (tid == 0) e_med = m; }
    __syncthreads();
    mx = red[0];
#pragma unroll
    for (int k = 1; k < GROUP / 32; ++k) mx = fmaxf(mx, red[k]);
    int fix = FIX_BITS;
    if (!COUNT && G.max_cnt > 0) fix = min(29, max(FIX_BITS, 30 - (32 - __clz(G.max_cnt))));     // max_cnt < 2^(32 - clz)
    int ex = 0;
    if (mx > 0.f) frexpf(mx, &ex);                               // every finite |c_i| < 2^ex
    if (e_med >= 0) ex = min(ex, e_med - 117);                   // 512 x the median's binade [2^(e-127), 2^(e-126))
    ex = max(ex, fix - 126);                                     // keeps both scales normal FP32 numbers
    const float scale = exp2f((float)(fix - ex)), inv_scale = exp2f((float)(ex - fix));
    const bool late = has && !(aci < ldexpf(1.f, ex));           // beyond the cap, Inf or NaN
    unsigned my_max = 0u;
    const int cfix = late ? 0 : __float2int_rn(ci * scale);

    // a late member's Delta contributions go straight to the global accumulator (its visits are counted in the window by
    // pass 2); done before pass 2, out of line, so that nothing of it stays live across the hot loop
    if (late) late_walk(g.sx, g.sy, g.sz, codes, code_off[i], start[i], n_vis, ci, COUNT ? &ds[0].x : dsum, COUNT ? 2 : 1);
    // ---- pass 2: {Delta, s} += {c_i, 1} on every visit; flush per slab -------------------------------------------------
    p = win_s + p_init + (COUNT ? 0u : (unsigned)(tid & 1) * (WIN_SLOTS * 4));     // odd lanes: second Delta copy
    w_next = __ldg(my_stream);
    c_next = (int)__ldg(my_cnt);
    for (int s = 0; s < G.nslab; ++s) {
        const int cmax = __reduce_max_sync(0xffffffffu, c_next);
        const unsigned long long w0 = w_next;
        if (s + 1 < G.nslab) {
            w_next = __ldg(my_stream + (size_t)(s + 1) * G.wps * GROUP);
            c_next = (int)__ldg(my_cnt + (size_t)(s + 1) * GROUP);
        }
        if (COUNT) {
            walk_slab(my_stream + (size_t)s * G.wps * GROUP, w0, cmax, tbl_s, p, [&](unsigned q) {
                const unsigned a = win_addr(q);
                atoms_add(a, cfix);
                atoms_inc(a + WIN_SLOTS * 4);
            });
        } else {
            walk_slab(my_stream + (size_t)s * G.wps * GROUP, w0, cmax, tbl_s, p, [&](unsigned q) { atoms_add(win_addr(q), cfix); });
        }
        __syncthreads();
        {
            const Column col = slab_column(G, wg, s, col_nq, col_ml);
            for_visited_slots(G, col, col_zq0, col_a0, wg.dim_z, [&](int z, unsigned a) {
                int* d0 = reinterpret_cast<int*>(win + a);
                unsigned* d1 = reinterpret_cast<unsigned*>(win + WIN_SLOTS * 4 + a);
                if (COUNT) {
                    const unsigned cs = *d1;
                    my_max = max(my_max, cs);
                    if (cs != 0u) {                   // a touched slot is a verified visit: it lies inside the grid
                        red_add_v2_w(ds + col.base + z * wg.stride_z, (float)*d0 * inv_scale, (float)cs);
                        *d0 = 0; *d1 = 0u;
                    }
                } else {
                    const int a0 = *d0, a1 = (int)*d1;
                    if ((a0 | a1) != 0) {             // only visited slots can be non-zero
                        if (a0 + a1 != 0) red_add_f32(dsum + col.base + z * wg.stride_z, (float)(a0 + a1) * inv_scale);
                        *d0 = 0; *d1 = 0u;
                    }
                }
            });
        }
        __syncthreads();
    }
    if (COUNT) {        // remember the largest slot count for the sweeps that reuse the cached counts
        my_max = __reduce_max_sync(0xffffffffu, my_max);
        if ((tid & 31) == 0 && my_max > 0u) atomicMax(&groups[launch_order[group0 + blockIdx.x]].max_cnt, (int)my_max);
    }
}

int launch_block_windowed(pct_ctx* ctx, const pct_paths* P, const SolvePlan* plan, int64_t block, bool count, const float* b,
                          const float* wts, const float* x, float2* ds, float* dsum, cudaStream_t st) {
    const int64_t g0 = plan->group_begin[(size_t)block], g1 = plan->group_begin[(size_t)block + 1];
    if (g1 <= g0) return PCT_OK;
    if (!ctx->k2w_ready) {
        PCT_CUDA(ctx, cudaFuncSetAttribute(k_block_windowed<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, K2W_SMEM));
        PCT_CUDA(ctx, cudaFuncSetAttribute(k_block_windowed<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, K2W_SMEM));
        ctx->k2w_ready = true;
    }
    ProfScope prof(ctx, 1, st);
    if (count)
        k_block_windowed<true><<<(unsigned)(g1 - g0), GROUP, K2W_SMEM, st>>>(ctx->cfg, P->N, P->ell, P->start, P->code_off, P->codes, plan->perm, plan->p0, plan->pflag,
                                                                            plan->cnt, plan->stream, plan->groups, plan->launch_order, g0, b, wts, x, ds, dsum);
    else
        k_block_windowed<false><<<(unsigned)(g1 - g0), GROUP, K2W_SMEM, st>>>(ctx->cfg, P->N, P->ell, P->start, P->code_off, P->codes, plan->perm, plan->p0, plan->pflag,
                                                                             plan->cnt, plan->stream, plan->groups, plan->launch_order, g0, b, wts, x, ds, dsum);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

}  // namespace pct
