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

constexpr int K2W_SMEM = WIN_SLOTS * 8;      // pass 1: float x[8192] in the first half; pass 2: int Delta[8192], uint s[8192]
constexpr int FIX_BITS = 17;                 // |c_i| 2^e < 2^17; <= MAX_ROW_VISITS * GROUP = 6144 additions per slot < 2^31

__device__ __forceinline__ void red_add_v2_w(float2* p, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

struct WinGeom {
    int dir, stride_m, stride_n, stride_z, dim_m, dim_n, dim_z;
    bool x_major;
};

// slot k of thread tid in a slab -> (nq, ml, zq).  The lane index runs along the grid's x axis (the contiguous one):
// the minor axis for y-major groups, the row (major) axis for x-major groups.
__device__ __forceinline__ void slot_coords(const WinGeom& w, int lin, int& nq, int& ml, int& zq) {
    if (w.x_major) { ml = lin & (SLAB - 1); nq = (lin >> 4) & (WIN_N - 1); }
    else { nq = lin & (WIN_N - 1); ml = (lin >> 5) & (SLAB - 1); }
    zq = lin >> 9;
}

// voxel index of window slot (nq, ml, zq) of slab s, or -1 if it lies outside the grid
__device__ __forceinline__ int slot_voxel(const PlanGroup& G, const WinGeom& w, int s, int nq, int ml, int zq) {
    const int r = s * SLAB + ml;
    const int nb = plan_nbase(G, r), zb = plan_zbase(G, r);
    const int n = nb + ((nq - nb) & (WIN_N - 1));
    const int z = zb + ((zq - zb) & (WIN_Z - 1));
    const int mj = G.m_first + w.dir * r;
    if ((unsigned)n >= (unsigned)w.dim_n || (unsigned)z >= (unsigned)w.dim_z || (unsigned)mj >= (unsigned)w.dim_m) return -1;
    return mj * w.stride_m + n * w.stride_n + z * w.stride_z;
}

struct Walker {
    const unsigned long long* cp;
    unsigned long long w;
    unsigned p;
    int nrem;
    // the first visit has no code: it is presented as one pad code (table entry 7 = no move)
    __device__ __forceinline__ void init(const unsigned long long* codes, unsigned p0) { cp = codes; w = 7ull; nrem = 1; p = p0; }
};

__global__ void __launch_bounds__(GROUP, 2)
k_block_windowed(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N, const float* __restrict__ ell,
                 const uint64_t* __restrict__ code_off, const ulonglong2* __restrict__ codes, const uint32_t* __restrict__ perm,
                 const uint32_t* __restrict__ p0, const uint8_t* __restrict__ pflag, const uint8_t* __restrict__ cnt,
                 const PlanGroup* __restrict__ groups, int64_t group0, const float* __restrict__ b, const float* __restrict__ x,
                 float2* __restrict__ ds) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ int2 tbl[8];
    __shared__ float red[GROUP / 32];
    __shared__ PlanGroup Gs;
    if (threadIdx.x == 0) Gs = groups[group0 + blockIdx.x];
    __syncthreads();
    const PlanGroup& G = Gs;
    if (G.cls == 7 || G.nslab == 0) return;
    const int tid = threadIdx.x;
    WinGeom wg;
    wg.x_major = G.cls < 2;
    wg.dir = (G.cls & 1) ? -1 : 1;
    wg.stride_m = wg.x_major ? 1 : g.nx; wg.stride_n = wg.x_major ? g.nx : 1; wg.stride_z = g.nx * g.ny;
    wg.dim_m = wg.x_major ? g.nx : g.ny; wg.dim_n = wg.x_major ? g.ny : g.nx; wg.dim_z = g.nz;
    if (tid < 8) {
        // {delta, field mask} of a step: fields are n (bits 2-6), row (7-10), z (11-14); additions wrap inside a field
        const int n_plus = wg.x_major ? 2 : 0;
        int2 e = make_int2(0, 0);
        if (tid == G.cls) e = make_int2(0x80, 0x780);
        else if (tid == n_plus) e = make_int2(0x4, 0x7C);
        else if (tid == n_plus + 1) e = make_int2(0x7C, 0x7C);
        else if (tid == 4) e = make_int2(0x800, 0x7800);
        else if (tid == 5) e = make_int2(0x7800, 0x7800);
        tbl[tid] = e;
    }
    const bool active = (uint32_t)tid < G.size && pflag[G.start + tid] != 0;
    uint32_t i = 0, n_vis = 0;
    unsigned p_init = 0;
    const unsigned long long* cp0 = nullptr;
    if (active) {
        i = perm[G.start + tid];
        n_vis = N[i];
        p_init = p0[G.start + tid];
        cp0 = reinterpret_cast<const unsigned long long*>(codes + code_off[i]);
    }
    const uint8_t* my_cnt = cnt + G.cnt_off + tid;
    float* xs = reinterpret_cast<float*>(smem);

    // ---- pass 1: S_i = sum of x over the visits ----------------------------------------------------------------------
    Walker wk;
    wk.init(cp0, p_init);
    float S = 0.f;
    for (int s = 0; s < G.nslab; ++s) {
        __syncthreads();                          // previous slab's walkers are done (and tbl is visible)
#pragma unroll
        for (int k = 0; k < WIN_SLOTS / GROUP; ++k) {
            int nq, ml, zq;
            slot_coords(wg, tid + k * GROUP, nq, ml, zq);
            const int vox = slot_voxel(G, wg, s, nq, ml, zq);
            xs[win_addr(win_pack(nq, ml, zq)) >> 2] = vox >= 0 ? __ldg(x + vox) : 0.f;
        }
        __syncthreads();
        int c = active ? (int)my_cnt[(size_t)s * GROUP] : 0;
        while (c > 0) {
            if (wk.nrem == 0) { wk.w = __ldg(wk.cp++); wk.nrem = CODES_PER_WORD; }
            int take = min(c, wk.nrem);
            c -= take; wk.nrem -= take;
            for (; take > 0; --take) {
                const int2 t = tbl[(unsigned)wk.w & 7u];
                wk.w >>= 3;
                wk.p = ((wk.p + (unsigned)t.x) & (unsigned)t.y) | (wk.p & ~(unsigned)t.y);
                S += *reinterpret_cast<const float*>(smem + win_addr(wk.p));
            }
        }
    }
    // ---- c_i and the CTA's fixed-point scale (R17, R21) -----------------------------------------------------------------
    float ci = 0.f;
    if (active && n_vis > 0) {
        const float l = ell[i];
        ci = (b[i] - l * S) / ((float)n_vis * l);
    }
    float mx = fabsf(ci);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    __syncthreads();                              // all walkers done with xs
    if ((tid & 31) == 0) red[tid >> 5] = mx;
    int* dl = reinterpret_cast<int*>(smem);
    unsigned* sc = reinterpret_cast<unsigned*>(smem + WIN_SLOTS * 4);
#pragma unroll
    for (int k = 0; k < 2 * WIN_SLOTS / GROUP; ++k) dl[tid + k * GROUP] = 0;      // clears Delta and s
    __syncthreads();
    mx = red[0];
#pragma unroll
    for (int k = 1; k < GROUP / 32; ++k) mx = fmaxf(mx, red[k]);
    int ex = 0;
    if (mx > 0.f && mx < INFINITY) frexpf(mx, &ex);              // mx < 2^ex
    const float scale = exp2f((float)(FIX_BITS - ex)), inv_scale = exp2f((float)(ex - FIX_BITS));
    const int cfix = __float2int_rn(ci * scale);

    // ---- pass 2: {Delta, s} += {c_i, 1} on every visit; flush per slab -------------------------------------------------
    wk.init(cp0, p_init);
    for (int s = 0; s < G.nslab; ++s) {
        int c = active ? (int)my_cnt[(size_t)s * GROUP] : 0;
        while (c > 0) {
            if (wk.nrem == 0) { wk.w = __ldg(wk.cp++); wk.nrem = CODES_PER_WORD; }
            int take = min(c, wk.nrem);
            c -= take; wk.nrem -= take;
            for (; take > 0; --take) {
                const int2 t = tbl[(unsigned)wk.w & 7u];
                wk.w >>= 3;
                wk.p = ((wk.p + (unsigned)t.x) & (unsigned)t.y) | (wk.p & ~(unsigned)t.y);
                const unsigned a = win_addr(wk.p);
                atomicAdd(reinterpret_cast<int*>(smem + a), cfix);
                atomicAdd(reinterpret_cast<unsigned*>(smem + WIN_SLOTS * 4 + a), 1u);
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < WIN_SLOTS / GROUP; ++k) {
            int nq, ml, zq;
            slot_coords(wg, tid + k * GROUP, nq, ml, zq);
            const unsigned a = win_addr(win_pack(nq, ml, zq)) >> 2;
            const unsigned cs = sc[a];
            if (cs != 0u) {
                const int vox = slot_voxel(G, wg, s, nq, ml, zq);
                red_add_v2_w(ds + vox, (float)dl[a] * inv_scale, (float)cs);
                dl[a] = 0; sc[a] = 0u;
            }
        }
        __syncthreads();
    }
}

int launch_block_windowed(pct_ctx* ctx, const pct_paths* P, const SolvePlan* plan, int64_t block, const float* b,
                          const float* x, float2* ds, cudaStream_t st) {
    const int64_t g0 = plan->group_begin[(size_t)block], g1 = plan->group_begin[(size_t)block + 1];
    if (g1 <= g0) return PCT_OK;
    if (!ctx->k2w_ready) {
        PCT_CUDA(ctx, cudaFuncSetAttribute(k_block_windowed, cudaFuncAttributeMaxDynamicSharedMemorySize, K2W_SMEM));
        ctx->k2w_ready = true;
    }
    ProfScope prof(ctx, 1, st);
    k_block_windowed<<<(unsigned)(g1 - g0), GROUP, K2W_SMEM, st>>>(ctx->cfg, P->N, P->ell, P->code_off, P->codes, plan->perm,
                                                                  plan->p0, plan->pflag, plan->cnt, plan->groups, g0, b, x, ds);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

}  // namespace pct
