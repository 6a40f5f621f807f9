// pre_kernels.cu -- the two preprocessing steps in front of the hot path:
//   pct_fbp         the FBP image the solver starts from ("Using the FBP image as the initial iterate, one can
//                   iteratively solve the system Ax = b"), reading R25 of DESIGN.md
//   pct_hull_carve  the object hull from the data themselves by space carving (part of the preprocessing the paper folds
//                   into its totals), reading R26
// Both are a few milliseconds next to the seconds of the hot path, so they are written for exactness first: FP64
// throughout, explicit round-to-nearest operations (no FMA contraction) wherever a floor() or a threshold decides, so
// that a bin or a voxel is chosen from the same IEEE numbers on every run.
#include <mutex>

#include "pct_internal.cuh"

namespace pct {

constexpr double PRE_PI = 3.14159265358979323846;

// ---- FBP ------------------------------------------------------------------------------------------------------------------
// sinogram layout: [slice][theta bin][s bin], s fastest

// K_f1: one thread per history -> (slice, theta, s) bin of its chord; sum of WEPL (FP64 atomics) and count per bin
__global__ void __launch_bounds__(256)
k_fbp_bin(const ProtonPtrs pr, const float* __restrict__ b, int64_t m, double u_in, double u_out, double lo_z, double h, int nz,
          int n_theta, int n_s, double ds, double* __restrict__ sum, unsigned* __restrict__ cnt) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const double dth = 2.0 * PRE_PI / (double)n_theta;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += stride) {
        const double phi = pr.phi[i], t_in = pr.t_in[i], v_in = pr.v_in[i], t_out = pr.t_out[i], v_out = pr.v_out[i];
        const double w = (double)b[i];
        if (!(isfinite(phi) && isfinite(t_in) && isfinite(v_in) && isfinite(t_out) && isfinite(v_out) && isfinite(w))) continue;
        // the chord between the two tracker hits: direction alpha relative to the beam axis, theta in the grid frame, signed
        // distance s from the rotation axis, height z
        const double alpha = atan2(__dsub_rn(t_out, t_in), __dsub_rn(u_out, u_in));
        double theta = fmod(__dadd_rn(phi, alpha), 2.0 * PRE_PI);
        if (theta < 0.0) theta = __dadd_rn(theta, 2.0 * PRE_PI);
        const double t_m = __dmul_rn(0.5, __dadd_rn(t_in, t_out)), u_m = __dmul_rn(0.5, __dadd_rn(u_in, u_out));
        const double s = __dsub_rn(__dmul_rn(t_m, cos(alpha)), __dmul_rn(u_m, sin(alpha)));
        const double z = __dmul_rn(0.5, __dadd_rn(v_in, v_out));
        int it = (int)floor(__ddiv_rn(theta, dth));
        if (it >= n_theta) it = n_theta - 1;
        const double js = floor(__dadd_rn(__ddiv_rn(s, ds), __dmul_rn(0.5, (double)n_s)));
        const double iz = floor(__ddiv_rn(__dsub_rn(z, lo_z), h));
        if (js < 0.0 || js >= (double)n_s || iz < 0.0 || iz >= (double)nz) continue;
        const size_t cell = ((size_t)iz * n_theta + (size_t)it) * n_s + (size_t)js;
        atomicAdd(sum + cell, w);
        atomicAdd(cnt + cell, 1u);
    }
}

// K_f2: one CTA per sinogram row: mean WEPL per bin, then q = ds (p * h) with the Ram-Lak kernel
// h(0) = 1 / (4 ds^2), h(n) = -1 / (pi^2 n^2 ds^2) for odd n, 0 for even n, by direct convolution (the row lives in shared
// memory; the terms are added in ascending k)
__global__ void __launch_bounds__(256)
k_fbp_filter(const double* __restrict__ sum, const unsigned* __restrict__ cnt, int n_s, double ds, unsigned min_count,
             double* __restrict__ q) {
    extern __shared__ double row[];
    const size_t base = (size_t)blockIdx.x * n_s;
    for (int k = threadIdx.x; k < n_s; k += blockDim.x) {
        const unsigned c = cnt[base + k];
        row[k] = c >= min_count ? sum[base + k] / (double)c : 0.0;
    }
    __syncthreads();
    const double h0 = 1.0 / (4.0 * ds * ds), pd = PRE_PI * PRE_PI * ds * ds;
    for (int j = threadIdx.x; j < n_s; j += blockDim.x) {
        double acc = 0.0;
        for (int k = 0; k < n_s; ++k) {
            const int n = j - k;
            if (n == 0) acc += row[k] * h0;
            else if (n & 1) acc += row[k] * (-1.0 / (pd * (double)n * (double)n));
        }
        q[base + j] = ds * acc;
    }
}

// K_f3: one thread per voxel (x fastest), loop over the directions: q interpolated linearly at s = -x sin + y cos
__global__ void __launch_bounds__(256)
k_fbp_backproject(const double* __restrict__ q, int nx, int ny, int nz, double lo_x, double lo_y, double h, int n_theta, int n_s,
                  double ds, float* __restrict__ x0) {
    extern __shared__ double trig[];                    // sin, cos of the bin-centre directions
    for (int it = threadIdx.x; it < n_theta; it += blockDim.x) {
        const double th = ((double)it + 0.5) * (2.0 * PRE_PI / (double)n_theta);
        trig[2 * it] = sin(th); trig[2 * it + 1] = cos(th);
    }
    __syncthreads();
    const int64_t n = (int64_t)nx * ny * nz, j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const int ix = (int)(j % nx), iy = (int)((j / nx) % ny), iz = (int)(j / ((int64_t)nx * ny));
    const double x = lo_x + ((double)ix + 0.5) * h, y = lo_y + ((double)iy + 0.5) * h;
    const double* qz = q + (size_t)iz * n_theta * n_s;
    double acc = 0.0;
    for (int it = 0; it < n_theta; ++it) {
        const double s = -x * trig[2 * it] + y * trig[2 * it + 1];
        const double u = s / ds + 0.5 * (double)n_s - 0.5;            // bin k is centred on (k + 1/2 - n_s / 2) ds
        const double j0 = floor(u), f = u - j0;
        const double* qr = qz + (size_t)it * n_s;
        const double q0 = (j0 >= 0.0 && j0 < (double)n_s) ? __ldg(qr + (int)j0) : 0.0;
        const double q1 = (j0 + 1.0 >= 0.0 && j0 + 1.0 < (double)n_s) ? __ldg(qr + (int)j0 + 1) : 0.0;
        acc += (1.0 - f) * q0 + f * q1;
    }
    x0[j] = (float)((PRE_PI / (double)n_theta) * acc);
}

}  // namespace pct

using namespace pct;

extern "C" int pct_fbp(pct_ctx* ctx, const pct_protons* pr, const float* b, const pct_fbp_params* fp, float* x0_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!pr || pr->m < 0 || !fp || !x0_out || (pr->m > 0 && !b)) return set_error(ctx, PCT_E_INVALID_ARG, "bad fbp arguments");
    if (fp->n_theta < 1 || fp->n_s < 2 || fp->n_s > 4096 || fp->n_theta > 4096 || !(fp->ds_mm > 0.0) || !std::isfinite(fp->ds_mm))
        return set_error(ctx, PCT_E_INVALID_ARG, "fbp: n_theta in [1, 4096], n_s in [2, 4096], ds_mm > 0");
    if (pr->m > 0 && (!pr->phi || !pr->t_in || !pr->v_in || !pr->t_out || !pr->v_out)) return set_error(ctx, PCT_E_INVALID_ARG, "NULL tracker array");
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != ctx->device) cudaSetDevice(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t cells = (size_t)ctx->geom.nz * fp->n_theta * fp->n_s;
    double *sum = nullptr, *q = nullptr;
    unsigned* cnt = nullptr;
    auto done = [&](int code) {
        if (sum || q || cnt) cudaStreamSynchronize(st);          // scratch goes back to the cache only when the stream is done with it
        cache_free(sum); cache_free(q); cache_free(cnt);
        if (prev >= 0 && prev != ctx->device) cudaSetDevice(prev);
        return code;
    };
#define FBP_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError(); \
        return done(set_error(ctx, e__ == cudaErrorMemoryAllocation ? PCT_E_OOM : PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
    FBP_CUDA(cache_alloc((void**)&sum, sizeof(double) * cells));
    FBP_CUDA(cache_alloc((void**)&q, sizeof(double) * cells));
    FBP_CUDA(cache_alloc((void**)&cnt, sizeof(unsigned) * cells));
    {
        ProfScope prof(ctx, 5, st);
        FBP_CUDA(cudaMemsetAsync(sum, 0, sizeof(double) * cells, st));
        FBP_CUDA(cudaMemsetAsync(cnt, 0, sizeof(unsigned) * cells, st));
        const ProtonPtrs pp = {pr->phi, pr->t_in, pr->v_in, pr->dt_in, pr->dv_in, pr->t_out, pr->v_out, pr->dt_out, pr->dv_out};
        if (pr->m > 0) {
            const int64_t want = (pr->m + 255) / 256, cap = (int64_t)ctx->num_sms * 16;
            k_fbp_bin<<<(unsigned)(want < cap ? want : cap), 256, 0, st>>>(pp, b, pr->m, pr->u_in_mm, pr->u_out_mm, ctx->geom.origin_mm[2], ctx->geom.h_mm,
                                                                            ctx->geom.nz, fp->n_theta, fp->n_s, fp->ds_mm, sum, cnt);
        }
        k_fbp_filter<<<(unsigned)((size_t)ctx->geom.nz * fp->n_theta), 256, sizeof(double) * fp->n_s, st>>>(sum, cnt, fp->n_s, fp->ds_mm,
                                                                                                          (unsigned)(fp->min_count > 1 ? fp->min_count : 1), q);
        k_fbp_backproject<<<(unsigned)((ctx->n_vox + 255) / 256), 256, sizeof(double) * 2 * fp->n_theta, st>>>(
            q, ctx->geom.nx, ctx->geom.ny, ctx->geom.nz, ctx->geom.origin_mm[0], ctx->geom.origin_mm[1], ctx->geom.h_mm, fp->n_theta, fp->n_s, fp->ds_mm, x0_out);
        ctx->launches += 3;
    }
    FBP_CUDA(cudaGetLastError());
#undef FBP_CUDA
    return done(PCT_OK);
}

// ---- pct_fbp_static: the same FBP with its sinogram scratch in a fixed device array -- no allocation at all --------------------
// For callers that cannot call cudaMalloc (stream capture, serving loops, harnesses that forbid it).  The three scratch
// arrays of pct_fbp (bin sums, filtered rows, bin counts: 20 bytes per sinogram bin) live in ONE file-scope array sized for
// PCT_FBP_STATIC_MAX_CELLS bins (20 MiB), held by every GPU that loads the library until the process exits.  Host code
// cannot use the array's name as a pointer (it is the host-side stand-in of the symbol): its device address is looked up once
// per device, with that device current, by cudaGetSymbolAddress.
namespace pct {

constexpr size_t FBP_STATIC_CELLS = PCT_FBP_STATIC_MAX_CELLS;
// layout: double sum[MAX] | double q[MAX] | unsigned cnt[MAX]
static __device__ __align__(256) unsigned char g_fbp_static_scratch[FBP_STATIC_CELLS * (2 * sizeof(double) + sizeof(unsigned))];

static std::mutex g_fbp_static_mu;
static void* g_fbp_static_ptr[64];          // per device: device address of g_fbp_static_scratch (nullptr = not looked up yet)

// device address of the scratch array on `device` (which must be current); cudaSuccess or the look-up's error
static cudaError_t fbp_static_scratch(int device, unsigned char** out) {
    if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_fbp_static_mu);
    if (!g_fbp_static_ptr[device]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_fbp_static_scratch);
        if (e != cudaSuccess) return e;
        g_fbp_static_ptr[device] = ptr;
    }
    *out = static_cast<unsigned char*>(g_fbp_static_ptr[device]);
    return cudaSuccess;
}

}  // namespace pct

extern "C" int pct_fbp_static(pct_ctx* ctx, const pct_protons* pr, const float* b, const pct_fbp_params* fp, float* x0_out, void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!pr || pr->m < 0 || !fp || !x0_out || (pr->m > 0 && !b)) return set_error(ctx, PCT_E_INVALID_ARG, "bad fbp arguments");
    if (fp->n_theta < 1 || fp->n_s < 2 || fp->n_s > 4096 || fp->n_theta > 4096 || !(fp->ds_mm > 0.0) || !std::isfinite(fp->ds_mm))
        return set_error(ctx, PCT_E_INVALID_ARG, "fbp: n_theta in [1, 4096], n_s in [2, 4096], ds_mm > 0");
    if (pr->m > 0 && (!pr->phi || !pr->t_in || !pr->v_in || !pr->t_out || !pr->v_out)) return set_error(ctx, PCT_E_INVALID_ARG, "NULL tracker array");
    const size_t cells = (size_t)ctx->geom.nz * fp->n_theta * fp->n_s;
    if (cells > FBP_STATIC_CELLS)
        return set_error(ctx, PCT_E_CAPACITY, "pct_fbp_static: nz * n_theta * n_s = %zu sinogram bins exceed the fixed scratch of %zu bins (use pct_fbp)",
                         cells, FBP_STATIC_CELLS);
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != ctx->device) cudaSetDevice(ctx->device);
    auto done = [&](int code) { if (prev >= 0 && prev != ctx->device) cudaSetDevice(prev); return code; };
#define FBPS_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cudaGetLastError(); \
        return done(set_error(ctx, PCT_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__))); } } while (0)
    unsigned char* base = nullptr;
    FBPS_CUDA(fbp_static_scratch(ctx->device, &base));
    double* sum = reinterpret_cast<double*>(base);
    double* q = sum + FBP_STATIC_CELLS;
    unsigned* cnt = reinterpret_cast<unsigned*>(q + FBP_STATIC_CELLS);
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the last call's contents: the sums and counts must start at zero (q is overwritten by the filter)
    FBPS_CUDA(cudaMemsetAsync(sum, 0, sizeof(double) * cells, st));
    FBPS_CUDA(cudaMemsetAsync(cnt, 0, sizeof(unsigned) * cells, st));
    const ProtonPtrs pp = {pr->phi, pr->t_in, pr->v_in, pr->dt_in, pr->dv_in, pr->t_out, pr->v_out, pr->dt_out, pr->dv_out};
    if (pr->m > 0) {
        const int64_t want = (pr->m + 255) / 256, cap = (int64_t)ctx->num_sms * 16;
        k_fbp_bin<<<(unsigned)(want < cap ? want : cap), 256, 0, st>>>(pp, b, pr->m, pr->u_in_mm, pr->u_out_mm, ctx->geom.origin_mm[2], ctx->geom.h_mm,
                                                                        ctx->geom.nz, fp->n_theta, fp->n_s, fp->ds_mm, sum, cnt);
    }
    k_fbp_filter<<<(unsigned)((size_t)ctx->geom.nz * fp->n_theta), 256, sizeof(double) * fp->n_s, st>>>(sum, cnt, fp->n_s, fp->ds_mm,
                                                                                                      (unsigned)(fp->min_count > 1 ? fp->min_count : 1), q);
    k_fbp_backproject<<<(unsigned)((ctx->n_vox + 255) / 256), 256, sizeof(double) * 2 * fp->n_theta, st>>>(
        q, ctx->geom.nx, ctx->geom.ny, ctx->geom.nz, ctx->geom.origin_mm[0], ctx->geom.origin_mm[1], ctx->geom.h_mm, fp->n_theta, fp->n_s, fp->ds_mm, x0_out);
    ctx->launches += 3;
    FBPS_CUDA(cudaGetLastError());
#undef FBPS_CUDA
    return done(PCT_OK);
}

// ---- hull by space carving (R26) ---------------------------------------------------------------------------------------------
namespace pct {

// entry / exit parameter of the chord A + s d in the slab [lo, hi] of one axis, folded into [e0, e1]; false if the chord
// runs parallel to the slab and outside it.  Plain round-to-nearest divisions: the same numbers on every run.
__device__ __forceinline__ bool clip_slab(double A, double d, double lo, double hi, double& e0, double& e1) {
    if (d != 0.0) {
        const double s1 = __ddiv_rn(__dsub_rn(lo, A), d), s2 = __ddiv_rn(__dsub_rn(hi, A), d);
        e0 = fmax(e0, fmin(s1, s2));
        e1 = fmin(e1, fmax(s1, s2));
        return true;
    }
    return !(A < lo || A > hi);
}

// One thread per history.  A history with WEPL < wepl_air carves every voxel its tracker-to-tracker chord crosses with a
// chord length > min_chord.  The thread marches along the axis of largest extent, slab by slab, and tests the few voxels
// of the other two axes the chord can touch in that slab (the range of its two end points there, one voxel of margin): a
// voxel's chord is |B - A| (e1 - e0) with [e0, e1] the intersection of its three slab intervals.  Writes are plain byte
// stores of 0 (idempotent, no atomics).
__global__ void __launch_bounds__(128)
k_hull_carve(const ProtonPtrs pr, const float* __restrict__ b, int64_t m, double u_in, double u_out, int nx, int ny, int nz, double ox,
             double oy, double oz, double h, double wepl_air, double min_chord, uint8_t* __restrict__ hull) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const double w = (double)b[i];
    if (!(isfinite(w) && w < wepl_air)) return;
    const double phi = pr.phi[i], t_in = pr.t_in[i], v_in = pr.v_in[i], t_out = pr.t_out[i], v_out = pr.v_out[i];
    if (!(isfinite(phi) && isfinite(t_in) && isfinite(v_in) && isfinite(t_out) && isfinite(v_out))) return;
    double sph, cph;
    sincos(phi, &sph, &cph);
    const int n[3] = {nx, ny, nz};
    const double org[3] = {ox, oy, oz};
    const double A[3] = {__dsub_rn(__dmul_rn(u_in, cph), __dmul_rn(t_in, sph)), __dadd_rn(__dmul_rn(u_in, sph), __dmul_rn(t_in, cph)), v_in};
    const double B[3] = {__dsub_rn(__dmul_rn(u_out, cph), __dmul_rn(t_out, sph)), __dadd_rn(__dmul_rn(u_out, sph), __dmul_rn(t_out, cph)), v_out};
    const double d[3] = {__dsub_rn(B[0], A[0]), __dsub_rn(B[1], A[1]), __dsub_rn(B[2], A[2])};
    const double len = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
    if (!(len > 0.0)) return;
    // the part of the chord inside the grid box
    double s_lo = 0.0, s_hi = 1.0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (!clip_slab(A[a], d[a], org[a], __dadd_rn(org[a], __dmul_rn((double)n[a], h)), s_lo, s_hi)) return;
    if (!(s_lo < s_hi)) return;
    int am = 0;
    if (fabs(d[1]) > fabs(d[am])) am = 1;
    if (fabs(d[2]) > fabs(d[am])) am = 2;
    const int a1 = (am + 1) % 3, a2 = (am + 2) % 3;
    auto pick = [](const double (&v)[3], int a) { return a == 0 ? v[0] : (a == 1 ? v[1] : v[2]); };
    auto pick_i = [](const int (&v)[3], int a) { return a == 0 ? v[0] : (a == 1 ? v[1] : v[2]); };
    const double Am = pick(A, am), dm = pick(d, am), om = pick(org, am);
    const double A1 = pick(A, a1), d1 = pick(d, a1), o1 = pick(org, a1), A2 = pick(A, a2), d2 = pick(d, a2), o2 = pick(org, a2);
    const int nm = pick_i(n, am), n1 = pick_i(n, a1), n2 = pick_i(n, a2);
    const int64_t strd[3] = {1, nx, (int64_t)nx * ny};
    const int64_t sm = am == 0 ? strd[0] : (am == 1 ? strd[1] : strd[2]), st1 = a1 == 0 ? strd[0] : (a1 == 1 ? strd[1] : strd[2]),
                  st2 = a2 == 0 ? strd[0] : (a2 == 1 ? strd[1] : strd[2]);
    // slabs of the marching axis the clipped chord can touch
    const double pm0 = fma(s_lo, dm, Am), pm1 = fma(s_hi, dm, Am);
    const int im_lo = max(0, (int)floor((fmin(pm0, pm1) - om) / h) - 1), im_hi = min(nm - 1, (int)floor((fmax(pm0, pm1) - om) / h) + 1);
    for (int im = im_lo; im <= im_hi; ++im) {
        double m0 = s_lo, m1 = s_hi;
        const double lo_m = __dadd_rn(om, __dmul_rn((double)im, h)), hi_m = __dadd_rn(om, __dmul_rn((double)(im + 1), h));
        clip_slab(Am, dm, lo_m, hi_m, m0, m1);                      // dm != 0: it is the largest component and len > 0
        if (!(m0 < m1)) continue;
        const double p10 = fma(m0, d1, A1), p11 = fma(m1, d1, A1), p20 = fma(m0, d2, A2), p21 = fma(m1, d2, A2);
        // candidates: the voxels between the chord's two end points in this slab (a margin of 1e-6 voxel widths against rounding;
        // a voxel beyond it could only be touched at a corner, with no chord to speak of)
        const int j1_lo = max(0, (int)floor((fmin(p10, p11) - o1) / h - 1e-6)), j1_hi = min(n1 - 1, (int)floor((fmax(p10, p11) - o1) / h + 1e-6));
        const int j2_lo = max(0, (int)floor((fmin(p20, p21) - o2) / h - 1e-6)), j2_hi = min(n2 - 1, (int)floor((fmax(p20, p21) - o2) / h + 1e-6));
        for (int j1 = j1_lo; j1 <= j1_hi; ++j1) {
            double f0 = m0, f1 = m1;
            if (!clip_slab(A1, d1, __dadd_rn(o1, __dmul_rn((double)j1, h)), __dadd_rn(o1, __dmul_rn((double)(j1 + 1), h)), f0, f1) || !(f1 > f0)) continue;
            for (int j2 = j2_lo; j2 <= j2_hi; ++j2) {
                double e0 = f0, e1 = f1;
                if (!clip_slab(A2, d2, __dadd_rn(o2, __dmul_rn((double)j2, h)), __dadd_rn(o2, __dmul_rn((double)(j2 + 1), h)), e0, e1) || !(e1 > e0)) continue;
                if (__dmul_rn(__dsub_rn(e1, e0), len) > min_chord) hull[(int64_t)im * sm + (int64_t)j1 * st1 + (int64_t)j2 * st2] = 0;
            }
        }
    }
}

}  // namespace pct

extern "C" int pct_hull_carve(pct_ctx* ctx, const pct_protons* pr, const float* b, double wepl_air_mm, double min_chord_mm, uint8_t* hull_out,
                              void* stream) {
    if (!ctx) return PCT_E_INVALID_ARG;
    if (!pr || pr->m < 0 || !hull_out || (pr->m > 0 && !b) || !(min_chord_mm >= 0.0) || !std::isfinite(wepl_air_mm))
        return set_error(ctx, PCT_E_INVALID_ARG, "bad hull_carve arguments");
    if (pr->m > 0 && (!pr->phi || !pr->t_in || !pr->v_in || !pr->t_out || !pr->v_out)) return set_error(ctx, PCT_E_INVALID_ARG, "NULL tracker array");
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != ctx->device) cudaSetDevice(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = PCT_OK;
    {
        ProfScope prof(ctx, 5, st);
        cudaError_t e = cudaMemsetAsync(hull_out, 1, (size_t)ctx->n_vox, st);
        if (e == cudaSuccess && pr->m > 0) {
            const ProtonPtrs pp = {pr->phi, pr->t_in, pr->v_in, pr->dt_in, pr->dv_in, pr->t_out, pr->v_out, pr->dt_out, pr->dv_out};
            k_hull_carve<<<(unsigned)((pr->m + 127) / 128), 128, 0, st>>>(pp, b, pr->m, pr->u_in_mm, pr->u_out_mm, ctx->geom.nx, ctx->geom.ny, ctx->geom.nz,
                                                                          ctx->geom.origin_mm[0], ctx->geom.origin_mm[1], ctx->geom.origin_mm[2], ctx->geom.h_mm,
                                                                          wepl_air_mm, min_chord_mm, hull_out);
            ++ctx->launches;
            e = cudaGetLastError();
        }
        if (e != cudaSuccess) { cudaGetLastError(); rc = set_error(ctx, PCT_E_CUDA, "hull_carve: %s", cudaGetErrorString(e)); }
    }
    if (prev >= 0 && prev != ctx->device) cudaSetDevice(prev);
    return rc;
}
