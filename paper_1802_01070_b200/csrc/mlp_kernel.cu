// mlp_kernel.cu -- K1: tracker record -> hull entry/exit (A1) -> most likely path (A2) -> voxel walk + 3-bit
// step codes (A3).  PAPER.md:7 ("calculating the individual proton's most likely path [3]" gives the rows of A),
// PAPER.md:26 ("each proton as an individual thread").  FP64 throughout; readings R1-R12 of DESIGN.md.
//
// Two kernels per batch of 2^20 histories, one thread per history: k_hull (hull entry/exit and the per-history part of the
// MLP) and k_mlp_walk (the MLP sample by sample, the voxel steps of every segment without a data-dependent loop).  Bound by
// instruction issue: ~90 FP64 instructions per MLP sample (K ~ 2*depth samples), each of which holds the issue port for
// two cycles on sm_100a, plus the bookkeeping of the walk; memory is irrelevant (72 B in, ~60-170 B out per history).
// Rows are copied to the code stream at a place taken from an atomic chunk counter.
#include <cub/device/device_radix_sort.cuh>

#include "pct_internal.cuh"

namespace pct {

__device__ __forceinline__ double face_coord(const DevCfg& g, int a, int i) { return fma((double)i, g.h, g.lo[a]); }

struct Hit { bool ok, tie; int c[3]; double P[3]; };

// A1 / R3-R4: from the tracker point T along d (not normalised) to the first hull voxel V_s and the point P_0 where the
// ray enters it.  Written as a ray-parameter traversal (Amanatides & Woo): the point is T + s d, s >= 0, and everything
// is expressed in s -- the interval [s_in, s_out] in which the ray is inside the search box, and per axis the parameter
// s_next[a] of the next voxel face.  The search box is the bounding box of the hull voxels (g.bmin..g.bmax; the whole
// grid if hull == NULL): a straight ray visits the same voxels wherever the traversal starts, so the air between the
// grid faces and that box is skipped.  Decisions (which face comes first) are those of rule R9 applied to the chord of
// the ray in the box; two faces closer than tie_eps along the ray set the tie flag.  Inside the loop s_next uses one
// reciprocal per axis; P_0 is computed from the exact quotient of the face that was crossed last.
__device__ __forceinline__ void find_hull(const DevCfg& g, const uint8_t* __restrict__ hull, const double (&T)[3],
                                       const double (&d)[3], Hit& hit) {
    hit.ok = false; hit.tie = false;
    const double d_len = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    const double tie_s = d_len > 0.0 ? g.tie_eps / d_len : 0.0;        // tie_eps (mm along the ray) as a parameter difference
    // per axis: the parameter interval in which the ray is between the box's two faces
    double s_in = 0.0, s_out = INFINITY, s_enter[3];
    int ax_in = -1;                                                    // axis through whose face the ray enters (-1: T is inside)
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double b_lo = face_coord(g, a, g.bmin[a]), b_hi = face_coord(g, a, g.bmax[a] + 1);
        s_enter[a] = -INFINITY;
        if (d[a] > 0.0) { s_enter[a] = (b_lo - T[a]) / d[a]; s_out = fmin(s_out, (b_hi - T[a]) / d[a]); }
        else if (d[a] < 0.0) { s_enter[a] = (b_hi - T[a]) / d[a]; s_out = fmin(s_out, (b_lo - T[a]) / d[a]); }
        else if (T[a] < b_lo || T[a] > b_hi) return;                   // parallel to this slab and outside it
        if (s_enter[a] > s_in) { s_in = s_enter[a]; ax_in = a; }
    }
    if (!(s_in < s_out)) return;                                       // the ray passes beside the box (or only touches it)
    // entry voxel: the boundary index on the entering axis, the voxel containing the entry point on the other two
    int c[3], step[3], left[3], dlin[3];
    double inv[3], s_next[3], P[3];
    const int stride[3] = {1, g.nx, g.nx * g.ny};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        step[a] = d[a] > 0.0 ? 1 : (d[a] < 0.0 ? -1 : 0);
        if (a == ax_in) {
            c[a] = step[a] > 0 ? g.bmin[a] : g.bmax[a];
            P[a] = face_coord(g, a, step[a] > 0 ? g.bmin[a] : g.bmax[a] + 1);         // on the face, exactly
        } else {
            if (ax_in >= 0 && s_in - s_enter[a] < tie_s) hit.tie = true;             // enters through an edge of the box
            P[a] = fma(s_in, d[a], T[a]);
            c[a] = min(max((int)floor((P[a] - g.lo[a]) / g.h), g.bmin[a]), g.bmax[a]);
        }
        left[a] = step[a] > 0 ? g.bmax[a] - c[a] : c[a] - g.bmin[a];                  // steps this axis may still take in the box
        dlin[a] = step[a] * stride[a];
        inv[a] = step[a] != 0 ? 1.0 / d[a] : 0.0;
    }
    int crossed = -1;                                                   // axis of the face crossed last (-1: none yet)
    if (hull != nullptr) {
        // a face is a candidate while the ray's exit point of the box lies strictly beyond it (rule R9 on the chord);
        // s_next[a] = +inf marks "no further face on this axis"
        double E[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            E[a] = fma(s_out, d[a], T[a]);
            const double f = face_coord(g, a, c[a] + (step[a] > 0 ? 1 : 0));
            const bool cand = step[a] > 0 ? E[a] > f : (step[a] < 0 ? E[a] < f : false);
            s_next[a] = cand ? (f - T[a]) * inv[a] : INFINITY;
        }
        int lin = c[0] + g.nx * (c[1] + g.ny * c[2]);
        while (hull[lin] == 0) {
            int ax = 0;
            double sb = s_next[0];
            if (s_next[1] < sb) { ax = 1; sb = s_next[1]; }                 // strict: x before y before z on equality
            if (s_next[2] < sb) { ax = 2; sb = s_next[2]; }
            if (sb == INFINITY) return;                                     // the chord ends without meeting the hull
            if ((ax != 0 && s_next[0] - sb < tie_s) || (ax != 1 && s_next[1] - sb < tie_s) || (ax != 2 && s_next[2] - sb < tie_s)) hit.tie = true;
            // advance across the face of axis `ax`: the axis' quantities are selected, stepped once and put back -- one
            // converged path for the lanes of a warp, whichever axis each of them steps along
            {
                const bool a0 = ax == 0, a1 = ax == 1;
                const int st = a0 ? step[0] : (a1 ? step[1] : step[2]);
                const int cn = (a0 ? c[0] : (a1 ? c[1] : c[2])) + st;
                const int lf = (a0 ? left[0] : (a1 ? left[1] : left[2])) - 1;
                if (lf < 0) return;                                        // left the hull's bounding box: miss
                lin += a0 ? dlin[0] : (a1 ? dlin[1] : dlin[2]);
                const double lo_a = a0 ? g.lo[0] : (a1 ? g.lo[1] : g.lo[2]), E_a = a0 ? E[0] : (a1 ? E[1] : E[2]);
                const double T_a = a0 ? T[0] : (a1 ? T[1] : T[2]), inv_a = a0 ? inv[0] : (a1 ? inv[1] : inv[2]);
                const double f = fma((double)(cn + (st > 0 ? 1 : 0)), g.h, lo_a);             // face_coord of the next face
                const bool cand = st > 0 ? E_a > f : E_a < f;
                const double sn = cand ? (f - T_a) * inv_a : INFINITY;
                c[0] = a0 ? cn : c[0]; c[1] = a1 ? cn : c[1]; c[2] = (a0 | a1) ? c[2] : cn;
                left[0] = a0 ? lf : left[0]; left[1] = a1 ? lf : left[1]; left[2] = (a0 | a1) ? left[2] : lf;
                s_next[0] = a0 ? sn : s_next[0]; s_next[1] = a1 ? sn : s_next[1]; s_next[2] = (a0 | a1) ? s_next[2] : sn;
            }
            crossed = ax;
        }
    }
    if (crossed >= 0) {
        // P_0 = the point of the ray on the face through which V_s was entered: exact quotient, exact face coordinate
        double face = 0.0, s_hit = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (a == crossed) { face = face_coord(g, a, c[a] + (step[a] > 0 ? 0 : 1)); s_hit = (face - T[a]) / d[a]; }
#pragma unroll
        for (int a = 0; a < 3; ++a) P[a] = a == crossed ? face : fma(s_hit, d[a], T[a]);
    } else if (ax_in < 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) P[a] = T[a];                            // the tracker point itself lies in a hull voxel
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) { hit.c[a] = c[a]; hit.P[a] = P[a]; }
    hit.ok = true;
}

// degree-5 polynomial, Estrin's scheme: the same five FMAs as Horner's rule but a dependent chain of three (x2 = x * x)
__device__ __forceinline__ double poly5(const double (&c)[6], double x, double x2) {
    const double p01 = fma(c[1], x, c[0]), p23 = fma(c[3], x, c[2]), p45 = fma(c[5], x, c[4]);
    return fma(fma(p45, x2, p23), x2, p01);
}

// 1 / d for a normal, positive d: hardware seed (2^-23) and three Newton steps; not correctly rounded (a few 1e-16), which
// is all the MLP needs (positions to ~1e-12 mm, R24)
__device__ __forceinline__ double rcp_newton(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    r = fma(r, fma(-d, r, 1.0), r);
    r = fma(r, fma(-d, r, 1.0), r);
    return fma(r, fma(-d, r, 1.0), r);
}

// Row writer: 16-byte chunks of 42 codes, field k at bits 3(k%21) of word k/21; unused fields are 7 (pad).  A code is
// inserted at the top of the 64-bit word being filled and the word shifted down by one field per push, so that after 21
// pushes the first code sits in field 0 (one funnel shift and one OR per code, no variable shifts); a full word is stored
// through a running pointer (the two words of a chunk are consecutive in memory).
struct CodeWriter {
    unsigned long long acc;       // word being filled
    int nc;                       // codes in it (0..20)
    unsigned long long *wp, *w0;  // next word to store; first word of the row
    __device__ __forceinline__ void init(ulonglong2* s) { acc = 0ull; nc = 0; wp = w0 = reinterpret_cast<unsigned long long*>(s); }
    __device__ __forceinline__ void push(int code) {
        acc = (acc >> 3) | ((unsigned long long)code << 60);
        if (++nc == CODES_PER_WORD) { *wp++ = acc; acc = 0ull; nc = 0; }
    }
    // n = 0, 1 or 2 codes at once (c1 first): one converged path for all lanes of a warp whatever their n -- the shift is
    // 3 n bits and the codes enter the upper 32-bit half only.  A pair that straddles a word boundary goes code by code.
    __device__ __forceinline__ void push_upto2(int c1, int c2, int n) {
        if (n == 2 && nc == CODES_PER_WORD - 1) { push(c1); push(c2); return; }
        const unsigned sh = 3u * (unsigned)n;
        const unsigned bits = n == 2 ? (unsigned)(c1 | (c2 << 3)) : (unsigned)c1;
        const unsigned ins = n == 0 ? 0u : bits << (n == 2 ? 25 : 28);
        acc = (acc >> sh) | ((unsigned long long)ins << 32);
        nc += n;
        if (nc == CODES_PER_WORD) { *wp++ = acc; acc = 0ull; nc = 0; }
    }
    // the last word (k < 21 codes: shifted down to field 0, the rest pads) and a pad word if the chunk is half full; -> chunks
    __device__ __forceinline__ int finish() {
        if (nc > 0) *wp++ = (acc >> (3 * (CODES_PER_WORD - nc))) | (~0ull << (3 * nc));
        if ((wp - w0) & 1) *wp++ = ~0ull;
        return (int)((wp - w0) >> 1);
    }
};

// What k_hull (A1) hands to the walk kernels, per history: hull entry/exit, the MLP end states in the gantry frame (R5),
// the number of MLP segments K (R8; K = 0: rejected) and everything of the MLP that depends on the history only.
struct alignas(16) HistRec {
    double pin[3], pout[3];           // P_0, P_K (grid frame, mm)
    double cph, sph;                  // gantry angle
    double u0, t0, v0, t2, v2, D;     // end states; D = u2 - u0
    double du;                        // D / K
    double dt_in, dv_in, nu_t, nu_v;  // entry slopes; exit minus entry slopes
    double log_du;                    // ln(du / X0): ln(k du / X0) = ln k + log_du, ln k tabulated (one log per history)
    double cq[3][6];                  // Sigma2 moments: J_q(d2) = int_0^d2 r^q f(D - r) dr = d2^(q+1) sum_j cq[q][j] d2^j
    int32_t vin, vout;                // V_s, V_e (linear voxel index)
    uint32_t K, flags;
    int32_t cin[3];                   // V_s as (ix, iy, iz)
    int32_t pad_;
};

// Spatial sort key of a history inside its batch: 2 mm cell of the entry tracker hit, v-major.  Neighbouring threads
// of k_hull then shoot neighbouring, near-parallel rays: the hull search of a warp takes nearly the same steps.  The key
// only orders the work; it has no influence on any result.
__global__ void __launch_bounds__(256)
k_hull_keys(const ProtonPtrs pr, int64_t i_base, int count, double t_lo, double v_lo, double inv_cell, int nt, int nv,
            uint32_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= count) return;
    const double t = pr.t_in[i_base + p], v = pr.v_in[i_base + p];
    uint32_t key = 0;
    if (isfinite(t) && isfinite(v)) {
        const int tc = min(max((int)((t - t_lo) * inv_cell), 0), nt - 1), vc = min(max((int)((v - v_lo) * inv_cell), 0), nv - 1);
        key = (uint32_t)vc * (uint32_t)nt + (uint32_t)tc;
    }
    keys[p] = key;
    vals[p] = (uint32_t)p;
}

// A1 / R3-R5: tracker record -> hull entry/exit and the per-history part of the MLP.  Thread q takes history
// p = order[q] (spatial order, k_hull_keys).  Also emits, in that order, the sort key K: the walk kernels run the batch in
// order of K (longest first), so that concurrently running warps have the same trip count.
__global__ void __launch_bounds__(128, 5)
k_hull(const __grid_constant__ DevCfg g, const ProtonPtrs pr, const uint8_t* __restrict__ hull, int64_t i_base, int count,
       const uint32_t* __restrict__ order, HistRec* __restrict__ recs, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= count) return;
    const int p = (int)order[q];
    const int64_t i = i_base + p;
    const double phi = pr.phi[i], t_in = pr.t_in[i], v_in = pr.v_in[i], dt_in = pr.dt_in[i], dv_in = pr.dv_in[i];
    const double t_out = pr.t_out[i], v_out = pr.v_out[i], dt_out = pr.dt_out[i], dv_out = pr.dv_out[i];
    HistRec* r = recs + p;
    uint32_t K = 0, flags = 0;
    do {
        if (!(isfinite(phi) && isfinite(t_in) && isfinite(v_in) && isfinite(dt_in) && isfinite(dv_in) &&
              isfinite(t_out) && isfinite(v_out) && isfinite(dt_out) && isfinite(dv_out))) {
            flags = PCT_REJ_NONFINITE; break;
        }
        double sph, cph;
        sincos(phi, &sph, &cph);
        // R4: entry ray, reversed exit ray (grid frame, R1)
        Hit h_in, h_out;
        {
            const double T[3] = {g.u_in * cph - t_in * sph, g.u_in * sph + t_in * cph, v_in};
            const double d[3] = {cph - dt_in * sph, sph + dt_in * cph, dv_in};
            find_hull(g, hull, T, d, h_in);
        }
        {
            const double T[3] = {g.u_out * cph - t_out * sph, g.u_out * sph + t_out * cph, v_out};
            const double d[3] = {-(cph - dt_out * sph), -(sph + dt_out * cph), -dv_out};
            find_hull(g, hull, T, d, h_out);
        }
        if (!h_in.ok || !h_out.ok) { flags = PCT_REJ_MISS; break; }
        if (h_in.tie || h_out.tie) flags |= PCT_TIE;
        // R5: MLP end states in the gantry frame
        const double u0 = h_in.P[0] * cph + h_in.P[1] * sph, u2 = h_out.P[0] * cph + h_out.P[1] * sph;
        const double D = u2 - u0;
        if (!(D > 0.0)) { flags = PCT_REJ_ORDER; break; }
        if (D > g.max_depth) { flags = PCT_REJ_DEPTH; break; }
        K = (uint32_t)max(1, (int)ceil(D / (g.step_frac * g.h) - 1e-9));     // R8
        const double du = D / (double)K;
#pragma unroll
        for (int a = 0; a < 3; ++a) { r->pin[a] = h_in.P[a]; r->pout[a] = h_out.P[a]; }
        r->cph = cph; r->sph = sph;
        r->u0 = u0; r->t0 = -h_in.P[0] * sph + h_in.P[1] * cph; r->v0 = h_in.P[2];
        r->t2 = -h_out.P[0] * sph + h_out.P[1] * cph; r->v2 = h_out.P[2];
        r->D = D; r->du = du;
        r->dt_in = dt_in; r->dv_in = dv_in; r->nu_t = dt_out - dt_in; r->nu_v = dv_out - dv_in;
        r->log_du = log(du / g.X0);
        {   // f(D - r) = sum_j c_j r^j (Taylor shift of the polynomial about the exit depth D); cq[q][j] = c_j / (j + q + 1)
            const double binom[6][6] = {{1, 0, 0, 0, 0, 0}, {1, 1, 0, 0, 0, 0}, {1, 2, 1, 0, 0, 0},
                                        {1, 3, 3, 1, 0, 0}, {1, 4, 6, 4, 1, 0}, {1, 5, 10, 10, 5, 1}};
            double Dp[6];
            Dp[0] = 1.0;
#pragma unroll
            for (int e = 1; e < 6; ++e) Dp[e] = Dp[e - 1] * D;
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                double cj = 0.0;
#pragma unroll
                for (int ii = j; ii < 6; ++ii) cj += g.a[ii] * binom[ii][j] * Dp[ii - j];
                if (j & 1) cj = -cj;
#pragma unroll
                for (int qq = 0; qq < 3; ++qq) r->cq[qq][j] = cj / (double)(j + qq + 1);
            }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) r->cin[a] = h_in.c[a];
        r->vin = h_in.c[0] + g.nx * (h_in.c[1] + g.ny * h_in.c[2]);
        r->vout = h_out.c[0] + g.nx * (h_out.c[1] + g.ny * h_out.c[2]);
    } while (false);
    r->K = K; r->flags = flags;
    keys[q] = K;
    vals[q] = (uint32_t)p;
}

// The per-history constants of the MLP in registers (both walk kernels)
struct MlpHist {
    double u0, t0, v0, t2, v2, D, du, dt_in, dv_in, nu_t, nu_v, log_du;
    double cq[3][6];
    __device__ __forceinline__ void load(const HistRec* __restrict__ r) {
        u0 = r->u0; t0 = r->t0; v0 = r->v0; t2 = r->t2; v2 = r->v2; D = r->D; du = r->du;
        dt_in = r->dt_in; dv_in = r->dv_in; nu_t = r->nu_t; nu_v = r->nu_v; log_du = r->log_du;
#pragma unroll
        for (int q = 0; q < 3; ++q)
#pragma unroll
            for (int j = 0; j < 6; ++j) cq[q][j] = r->cq[q][j];
    }
};

// A2 / R7: most likely lateral positions (t, v) at depth w1 = k du, 0 < k < K -- the Gaussian-conditioning form of the MLP
// of ref [3] (positions only):  y = mu + Sigma1 R1^T (R1 Sigma1 R1^T + Sigma2)^-1 (y2 - R1 mu),  mu = R0 y0.
// Sigma1 moments are polynomials in w1 (DevCfg::s1c), Sigma2 moments in d2 = D - w1 (MlpHist::cq); the two log terms
// are ln(w1 / X0) = ln k + ln(du / X0) and ln(d2 / X0) = ln(K - k) + ln(du / X0).
__device__ __forceinline__ void mlp_sample(const DevCfg& g, const MlpHist& H, const double* __restrict__ logk, int k, int K,
                                           double& w1, double& tk, double& vk) {
    w1 = (double)k * H.du;
    const double d2 = H.D - w1;
    const double l1 = fma(g.log_coeff, __ldg(logk + k) + H.log_du, 1.0), l2 = fma(g.log_coeff, __ldg(logk + (K - k)) + H.log_du, 1.0);
    const double g1 = l1 * l1, g2 = l2 * l2;
    const double w1_2 = w1 * w1, d2_2 = d2 * d2;
    const double gw = g1 * w1, gd = g2 * d2;
    const double C1 = gw * poly5(g.s1c[0], w1, w1_2);
    const double B1 = (gw * w1) * poly5(g.s1c[1], w1, w1_2);
    const double A1 = (gw * w1_2) * poly5(g.s1c[2], w1, w1_2);
    const double C2 = gd * poly5(H.cq[0], d2, d2_2);
    const double B2 = (gd * d2) * poly5(H.cq[1], d2, d2_2);
    const double A2 = (gd * d2_2) * poly5(H.cq[2], d2, d2_2);
    const double P0 = fma(d2, B1, A1), P1 = fma(d2, C1, B1);      // first row / col of Sigma1 R1^T
    const double S00 = fma(d2, P1, P0) + A2, S01 = P1 + B2, S11 = C1 + C2;
    const double inv_det = rcp_newton(fma(S00, S11, -(S01 * S01)));
    const double G00 = (P0 * S11 - B1 * S01) * inv_det, G01 = (B1 * S00 - P0 * S01) * inv_det;
    const double mu_t = fma(w1, H.dt_in, H.t0), mu_v = fma(w1, H.dv_in, H.v0);
    tk = mu_t + G00 * (H.t2 - fma(d2, H.dt_in, mu_t)) + G01 * H.nu_t;
    vk = mu_v + G00 * (H.v2 - fma(d2, H.dv_in, mu_v)) + G01 * H.nu_v;
}

// sqrt(q), q > 0, to ~1e-14 relative: FP32 reciprocal square root as the seed, one Newton step in FP64 (the polyline length
// only enters the FP32 mean chord l_i)
__device__ __forceinline__ double sqrt_fast(double q) {
    const double y = (double)rsqrtf((float)q);
    const double r = q * y;
    return fma(0.5 * y, fma(-r, r, q), r);
}

// ---- A2 + A3: one thread per history, the MLP sample by sample, rule R9 segment by segment ---------------------
// A segment A -> B of the polyline is at most ~0.7 voxel widths long (R8: du <= h / 2), so it crosses at most ONE face per
// axis.  The common path therefore has no loop and no data-dependent branch on the axis: per axis the state d_a in
// {-1, 0, +1} says whether B lies beyond a face of the current voxel, the (up to two) steps are ordered by their crossing
// parameters only when a lane really has two of them (three: general loop), the voxel and its faces move by predicated updates, and the
// step codes are pushed in crossing order.  All 32 lanes of a warp (32 histories of equal sample count, neighbours in space)
// run this path together.  A segment that is longer than a voxel on some axis, steps out of the grid or exceeds the row
// capacity takes the general loop instead (rule R9 step by step, as DESIGN.md states it) from the same, uncommitted state.
// Codes go to a staging row per thread and are copied to the code stream once the row's length is known (chunk_counter
// hands out its place).
__global__ void __launch_bounds__(128, 4)
k_mlp_walk(const __grid_constant__ DevCfg g, const HistRec* __restrict__ recs, const uint32_t* __restrict__ order,
           const double* __restrict__ logk, int64_t i_base, int count, ulonglong2* __restrict__ stage, ulonglong2* __restrict__ codes,
           unsigned long long* __restrict__ chunk_counter, uint64_t* __restrict__ code_off, uint32_t* __restrict__ Nout,
           int32_t* __restrict__ start_out, int32_t* __restrict__ end_out, float* __restrict__ ell_out, uint8_t* __restrict__ flags_out,
           GenStats* __restrict__ stats) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = q < count;
    unsigned flags = 0;
    unsigned N = 0, n_samples = 0, n_general = 0;
    if (active) {
        const int p = (int)order[count - 1 - q];      // longest first: the CTAs launched last are the cheapest (short tail)
        const int64_t i = i_base + p;
        const HistRec* rec = recs + p;
        flags = rec->flags;
        int32_t start_v = -1, end_v = -1;
        float ell = 0.f;
        int n_chunks = 0;
        ulonglong2* my_stage = stage + (size_t)q * (size_t)g.stage_chunks;
        const int K = (int)rec->K;
        if (K > 0) do {
            MlpHist H;
            H.load(rec);
            const double cph = rec->cph, sph = rec->sph;
            const int vout = rec->vout;
            // R9-R11 walk state: current voxel, its faces, the previous vertex
            int c0 = rec->cin[0], c1 = rec->cin[1], c2 = rec->cin[2];
            start_v = rec->vin;
            CodeWriter cw;
            cw.init(my_stage);
            double A0 = rec->pin[0], A1 = rec->pin[1], A2 = rec->pin[2];
            double lo0 = face_coord(g, 0, c0), hi0 = face_coord(g, 0, c0 + 1), lo1 = face_coord(g, 1, c1), hi1 = face_coord(g, 1, c1 + 1),
                   lo2 = face_coord(g, 2, c2), hi2 = face_coord(g, 2, c2 + 1);
            double cd0 = (double)c0, cd1 = (double)c1, cd2 = (double)c2;
            double L = 0.0;
            int n_vis = 1;
            bool tie = false, bad = false;
            for (int k = 1; k <= K; ++k) {
                double B0, B1, B2;
                if (k < K) {
                    double w1, tk, vk;
                    mlp_sample(g, H, logk, k, K, w1, tk, vk);
                    const double uk = H.u0 + w1;
                    B0 = uk * cph - tk * sph; B1 = uk * sph + tk * cph; B2 = vk;
                } else {
                    B0 = rec->pout[0]; B1 = rec->pout[1]; B2 = rec->pout[2];
                }
                const double e0 = B0 - A0, e1 = B1 - A1, e2 = B2 - A2;
                const double q2 = fma(e0, e0, fma(e1, e1, e2 * e2));
                const double seg_len = q2 > 0.0 ? sqrt_fast(q2) : 0.0;
                L += seg_len;
                // state of every axis: B beyond the high face, beyond the low face, inside (closed voxel: a point on a face is inside)
                const int d0 = B0 > hi0 ? 1 : (B0 < lo0 ? -1 : 0), d1 = B1 > hi1 ? 1 : (B1 < lo1 ? -1 : 0), d2 = B2 > hi2 ? 1 : (B2 < lo2 ? -1 : 0);
                const int n = (d0 & 1) + (d1 & 1) + (d2 & 1);
                const int t0 = c0 + d0, t1 = c1 + d1, t2 = c2 + d2;
                const bool plain = q2 < g.h * g.h &&                       // shorter than a voxel: one face per axis at most
                                   (unsigned)t0 < (unsigned)g.nx && (unsigned)t1 < (unsigned)g.ny && (unsigned)t2 < (unsigned)g.nz &&
                                   n_vis + n <= g.max_visits && n <= 2;      // three faces in one segment: rare, general rule
                if (plain) {
                    // n == 2: the two crossing axes a < b are (0,1), (0,2) or (1,2).  Crossing parameter of an axis: s = num / den,
                    // num = distance of A from the face, den = |B - A| on that axis; s_b < s_a <=> num_b den_a < num_a den_b, and the
                    // tie test (s_a - s_b) |B - A| < eps likewise without a quotient; on equality the lower axis goes first (R9)
                    bool b_first = false;
                    if (n == 2) {
                        const bool z0 = d0 == 0, b2 = d2 != 0;                    // a = z0 ? 1 : 0, b = b2 ? 2 : 1
                        const double fa = z0 ? (d1 > 0 ? hi1 : lo1) : (d0 > 0 ? hi0 : lo0), fb = b2 ? (d2 > 0 ? hi2 : lo2) : (d1 > 0 ? hi1 : lo1);
                        const double na = fabs(fa - (z0 ? A1 : A0)), nb = fabs(fb - (b2 ? A2 : A1));
                        const double aa = fabs(z0 ? e1 : e0), ab = fabs(b2 ? e2 : e1);
                        const double la = na * ab, lb = nb * aa;
                        b_first = lb < la;
                        if (fabs(la - lb) * seg_len < g.tie_eps * (aa * ab)) tie = true;
                    }
                    // codes in crossing order: 0:+x 1:-x 2:+y 3:-y 4:+z 5:-z
                    const int k0c = d0 < 0 ? 1 : 0, k1c = d1 < 0 ? 3 : 2, k2c = d2 < 0 ? 5 : 4;
                    const int ca = d0 != 0 ? k0c : (d1 != 0 ? k1c : k2c);          // the first crossing axis in index order
                    const int cb = d2 != 0 ? k2c : k1c;                            // n == 2: the other one
                    cw.push_upto2(b_first ? cb : ca, b_first ? ca : cb, n);
                    // move
                    // (no branch: the voxel index, kept as a double too, follows d, and both faces are recomputed from it with
                    // face_coord's own fma -- the same values, also for an axis that did not move)
                    c0 = t0; c1 = t1; c2 = t2;
                    cd0 += B0 > hi0 ? 1.0 : (B0 < lo0 ? -1.0 : 0.0);
                    cd1 += B1 > hi1 ? 1.0 : (B1 < lo1 ? -1.0 : 0.0);
                    cd2 += B2 > hi2 ? 1.0 : (B2 < lo2 ? -1.0 : 0.0);
                    lo0 = fma(cd0, g.h, g.lo[0]); hi0 = fma(cd0 + 1.0, g.h, g.lo[0]);
                    lo1 = fma(cd1, g.h, g.lo[1]); hi1 = fma(cd1 + 1.0, g.h, g.lo[1]);
                    lo2 = fma(cd2, g.h, g.lo[2]); hi2 = fma(cd2 + 1.0, g.h, g.lo[2]);
                    n_vis += n;
                } else {
                    // the general rule R9: while B is strictly outside the closed voxel, step across the candidate face with the
                    // smallest crossing parameter
                    ++n_general;
                    int c[3] = {c0, c1, c2};
                    double f_lo[3] = {lo0, lo1, lo2}, f_hi[3] = {hi0, hi1, hi2};
                    const double A[3] = {A0, A1, A2}, B[3] = {B0, B1, B2};
                    int dd[3] = {d0, d1, d2};
                    while ((dd[0] | dd[1] | dd[2]) != 0) {
                        int best = dd[0] != 0 ? 0 : (dd[1] != 0 ? 1 : 2);
                        if ((dd[0] != 0) + (dd[1] != 0) + (dd[2] != 0) > 1) {
                            double num[3], den[3];
#pragma unroll
                            for (int a = 0; a < 3; ++a) {
                                num[a] = fabs((dd[a] > 0 ? f_hi[a] : f_lo[a]) - A[a]);
                                den[a] = fabs(B[a] - A[a]);
                            }
                            double nb = best == 0 ? num[0] : num[1], db_ = best == 0 ? den[0] : den[1];
                            if (best == 0 && dd[1] != 0 && num[1] * db_ < nb * den[1]) { best = 1; nb = num[1]; db_ = den[1]; }
                            if (dd[2] != 0 && num[2] * db_ < nb * den[2]) { best = 2; nb = num[2]; db_ = den[2]; }
#pragma unroll
                            for (int a = 0; a < 3; ++a)
                                if (a != best && dd[a] != 0 && fabs(num[a] * db_ - nb * den[a]) * seg_len < g.tie_eps * (den[a] * db_)) tie = true;
                        }
                        const int nn[3] = {g.nx, g.ny, g.nz};
                        int code = 0;
                        bool inside = true;
#pragma unroll
                        for (int a = 0; a < 3; ++a)
                            if (a == best) {
                                c[a] += dd[a];
                                code = 2 * a + (dd[a] < 0 ? 1 : 0);
                                inside = (unsigned)c[a] < (unsigned)nn[a];
                                if (dd[a] > 0) { f_lo[a] = f_hi[a]; f_hi[a] = face_coord(g, a, c[a] + 1); }
                                else { f_hi[a] = f_lo[a]; f_lo[a] = face_coord(g, a, c[a]); }
                                dd[a] = B[a] > f_hi[a] ? 1 : (B[a] < f_lo[a] ? -1 : 0);
                            }
                        ++n_vis;
                        if (!inside || n_vis > g.max_visits) { flags = !inside ? PCT_REJ_LEFT_GRID : PCT_REJ_CAPACITY; bad = true; break; }
                        cw.push(code);
                    }
                    if (bad) break;
                    c0 = c[0]; c1 = c[1]; c2 = c[2];
                    cd0 = (double)c0; cd1 = (double)c1; cd2 = (double)c2;
                    lo0 = f_lo[0]; lo1 = f_lo[1]; lo2 = f_lo[2]; hi0 = f_hi[0]; hi1 = f_hi[1]; hi2 = f_hi[2];
                }
                A0 = B0; A1 = B1; A2 = B2;
            }
            if (bad) break;
            n_chunks = cw.finish();
            N = (unsigned)n_vis;
            n_samples = (unsigned)K;
            if (tie) flags |= PCT_TIE;
            end_v = c0 + g.nx * (c1 + g.ny * c2);
            if (end_v != vout) flags |= PCT_END_MISMATCH;                                                    // R10
            ell = (float)(L / (double)N);                                                                    // R11
        } while (false);
        if (N == 0) { n_chunks = 0; start_v = -1; end_v = -1; ell = 0.f; }
        flags &= 0xffu;
        unsigned long long off = 0ull;
        if (n_chunks > 0) {
            off = atomicAdd(chunk_counter, (unsigned long long)n_chunks);
            for (int k = 0; k < n_chunks; ++k) codes[off + k] = my_stage[k];
        }
        code_off[i] = off;
        Nout[i] = N;
        start_out[i] = start_v;
        end_out[i] = end_v;
        ell_out[i] = ell;
        flags_out[i] = (uint8_t)flags;
    }
    // statistics: one atomic per warp and counter
    const unsigned vis = __reduce_add_sync(0xffffffffu, N);
    const unsigned rej = __reduce_add_sync(0xffffffffu, (active && N == 0) ? 1u : 0u);
    const unsigned tie_n = __reduce_add_sync(0xffffffffu, (flags & PCT_TIE) ? 1u : 0u);
    const unsigned smp = __reduce_add_sync(0xffffffffu, n_samples);
    const unsigned gen = __reduce_add_sync(0xffffffffu, n_general);
    if ((threadIdx.x & 31) == 0) {
        if (smp) atomicAdd(&stats->total_samples, (unsigned long long)smp);
        if (vis) atomicAdd(&stats->total_visits, (unsigned long long)vis);
        if (rej) atomicAdd(&stats->n_rejected, (unsigned long long)rej);
        if (tie_n) atomicAdd(&stats->n_ties, (unsigned long long)tie_n);
        if (gen) atomicAdd(&stats->n_general, (unsigned long long)gen);
    }
}

// scratch of one batch: history records, sort keys/values (double buffered), cub temporary storage
struct BatchScratch {
    HistRec* recs;
    cub::DoubleBuffer<uint32_t> dk, dv;     // K-order sort (key = K, value = local index)
    void* sort_tmp;
    size_t sort_tmp_bytes;
};

// A1 of one batch: spatial sort -> k_hull.  Leaves the records in S.recs (batch-local order) and the K keys in S.dk / S.dv.
static int hull_stage(pct_ctx* ctx, const ProtonPtrs& pr, const uint8_t* hull, int64_t i_base, int count, cudaStream_t st, BatchScratch& S) {
    const int threads = 128;
    const int blocks = (count + threads - 1) / threads;
    size_t sort_tmp = 0;
    {
        cub::DoubleBuffer<uint32_t> dk(nullptr, nullptr), dv(nullptr, nullptr);
        PCT_CUDA(ctx, cub::DeviceRadixSort::SortPairs(nullptr, sort_tmp, dk, dv, count, 0, 32, st));
    }
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    const size_t arr = up(4 * (size_t)count);
    const size_t o_rec = 0, o_k0 = up(sizeof(HistRec) * (size_t)count), o_k1 = o_k0 + arr, o_v0 = o_k1 + arr, o_v1 = o_v0 + arr,
                 o_k2 = o_v1 + arr, o_k3 = o_k2 + arr, o_v2 = o_k3 + arr, o_v3 = o_v2 + arr, o_tmp = o_v3 + arr, total = o_tmp + up(sort_tmp);
    if (total > ctx->gen_scratch_bytes) {
        if (ctx->gen_scratch) PCT_CUDA(ctx, cudaFree(ctx->gen_scratch));
        ctx->gen_scratch = nullptr; ctx->gen_scratch_bytes = 0;
        PCT_CUDA(ctx, cudaMalloc(&ctx->gen_scratch, total));
        ctx->gen_scratch_bytes = total;
    }
    char* base = (char*)ctx->gen_scratch;
    S.recs = (HistRec*)(base + o_rec);
    S.dk = cub::DoubleBuffer<uint32_t>((uint32_t*)(base + o_k0), (uint32_t*)(base + o_k1));
    S.dv = cub::DoubleBuffer<uint32_t>((uint32_t*)(base + o_v0), (uint32_t*)(base + o_v1));
    S.sort_tmp = base + o_tmp; S.sort_tmp_bytes = sort_tmp;
    cub::DoubleBuffer<uint32_t> sk((uint32_t*)(base + o_k2), (uint32_t*)(base + o_k3)), sv((uint32_t*)(base + o_v2), (uint32_t*)(base + o_v3));
    {   // spatial order of the batch: 2 mm cells of the entry tracker plane
        const DevCfg& c = ctx->cfg;
        const double ex = fmax(fabs(c.lo[0]), fabs(c.hi[0])), ey = fmax(fabs(c.lo[1]), fabs(c.hi[1]));
        const double t_half = sqrt(ex * ex + ey * ey), cell = 2.0 * c.h;
        const int nt = (int)fmin(4096.0, ceil(2.0 * t_half / cell) + 1.0), nv = (int)fmin(4096.0, ceil((c.hi[2] - c.lo[2]) / cell) + 1.0);
        k_hull_keys<<<(count + 255) / 256, 256, 0, st>>>(pr, i_base, count, -t_half, c.lo[2], 1.0 / cell, nt, nv, sk.Current(), sv.Current());
        int bits = 1;
        while ((1LL << bits) < (long long)nt * nv) ++bits;
        PCT_CUDA(ctx, cub::DeviceRadixSort::SortPairs(S.sort_tmp, sort_tmp, sk, sv, count, 0, bits, st));
    }
    k_hull<<<blocks, threads, 0, st>>>(ctx->cfg, pr, hull, i_base, count, sv.Current(), S.recs, S.dk.Current(), S.dv.Current());
    ctx->launches += 3;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// One batch of K1: spatial sort -> k_hull -> sort by K -> k_mlp_walk.  `stage` holds count rows of stage_chunks chunks; the
// rows are copied to the code stream at places handed out by the device counter `chunk_counter`.
int launch_mlp_batch(pct_ctx* ctx, const ProtonPtrs& pr, const uint8_t* hull, int64_t i_base, int count, ulonglong2* stage,
                     unsigned long long* chunk_counter, pct_paths* P, cudaStream_t st) {
    const int threads = 128;
    const int blocks = (count + threads - 1) / threads;
    ProfScope prof(ctx, 0, st);
    BatchScratch S;
    int rc;
    if ((rc = hull_stage(ctx, pr, hull, i_base, count, st, S)) != PCT_OK) return rc;
    int key_bits = 1;
    while ((1 << key_bits) < ctx->logk_n) ++key_bits;                  // K < logk_n
    PCT_CUDA(ctx, cub::DeviceRadixSort::SortPairs(S.sort_tmp, S.sort_tmp_bytes, S.dk, S.dv, count, 0, key_bits, st));
    k_mlp_walk<<<blocks, threads, 0, st>>>(ctx->cfg, S.recs, S.dv.Current(), ctx->logk, i_base, count, stage, P->codes, chunk_counter,
                                           P->code_off, P->N, P->start, P->end, P->ell, P->flags, ctx->d_stats);
    ctx->launches += 2;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// A1 alone (pct_hull_intersect): the hull entry and exit voxels of a batch, -1 for a history that A1 rejects
__global__ void __launch_bounds__(256) k_extract_ends(const HistRec* __restrict__ recs, int count, int32_t* __restrict__ v_in, int32_t* __restrict__ v_out) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= count) return;
    const bool rej = (recs[p].flags & PCT_REJECT_MASK) != 0;
    v_in[p] = rej ? -1 : recs[p].vin;
    v_out[p] = rej ? -1 : recs[p].vout;
}

int launch_hull_batch(pct_ctx* ctx, const ProtonPtrs& pr, const uint8_t* hull, int64_t i_base, int count, int32_t* v_in, int32_t* v_out, cudaStream_t st) {
    ProfScope prof(ctx, 0, st);
    BatchScratch S;
    int rc;
    if ((rc = hull_stage(ctx, pr, hull, i_base, count, st, S)) != PCT_OK) return rc;
    k_extract_ends<<<(count + 255) / 256, 256, 0, st>>>(S.recs, count, v_in + i_base, v_out + i_base);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// ---- bounding box of the hull mask: box6 = {min x, min y, min z, max x, max y, max z} (pre-set to {n.., -1..}) --------
__global__ void __launch_bounds__(256) k_hull_bbox(const __grid_constant__ DevCfg g, const uint8_t* __restrict__ hull, int* __restrict__ box6) {
    const int64_t n = (int64_t)g.nx * g.ny * g.nz, stride = (int64_t)gridDim.x * blockDim.x;
    int lo[3] = {INT_MAX, INT_MAX, INT_MAX}, hi[3] = {-1, -1, -1};
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += stride) {
        if (hull[j]) {
            const int c[3] = {(int)(j % g.nx), (int)((j / g.nx) % g.ny), (int)(j / ((int64_t)g.nx * g.ny))};
#pragma unroll
            for (int a = 0; a < 3; ++a) { lo[a] = min(lo[a], c[a]); hi[a] = max(hi[a], c[a]); }
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = __reduce_min_sync(0xffffffffu, lo[a]);
        hi[a] = __reduce_max_sync(0xffffffffu, hi[a]);
        if ((threadIdx.x & 31) == 0 && hi[a] >= 0) { atomicMin(box6 + a, lo[a]); atomicMax(box6 + 3 + a, hi[a]); }
    }
}

int launch_hull_bbox(pct_ctx* ctx, const uint8_t* hull, int* d_box6, cudaStream_t st) {
    const int init[6] = {INT_MAX, INT_MAX, INT_MAX, -1, -1, -1};
    PCT_CUDA(ctx, cudaMemcpyAsync(d_box6, init, sizeof(init), cudaMemcpyHostToDevice, st));
    k_hull_bbox<<<ctx->num_sms * 8, 256, 0, st>>>(ctx->cfg, hull, d_box6);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// ---- exclusive scan uint32 -> uint64 (three passes; sizes here are at most a few hundred M) ---------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ unsigned long long block_exclusive_scan(unsigned long long v, unsigned long long* total) {
    __shared__ unsigned long long warp_sums[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    if (lane == 31) warp_sums[w] = incl;
    __syncthreads();
    unsigned long long pre = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < SCAN_THREADS / 32; ++k) {
        const unsigned long long s = warp_sums[k];
        if (k < w) pre += s;
        tot += s;
    }
    __syncthreads();
    *total = tot;
    return pre + incl - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tile_sums(const uint32_t* __restrict__ in, int64_t n,
                                                                 unsigned long long* __restrict__ sums) {
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
    unsigned long long v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const int64_t i = base + (int64_t)k * SCAN_THREADS + threadIdx.x;
        if (i < n) v += in[i];
    }
    unsigned long long tot;
    block_exclusive_scan(v, &tot);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(unsigned long long* sums, int64_t nb, unsigned long long base,
                                                            unsigned long long* total_out) {
    unsigned long long carry = base;
    for (int64_t b0 = 0; b0 < nb; b0 += SCAN_THREADS) {
        const int64_t i = b0 + threadIdx.x;
        const unsigned long long v = i < nb ? sums[i] : 0ull;
        unsigned long long tot;
        const unsigned long long ex = block_exclusive_scan(v, &tot);
        if (i < nb) sums[i] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry - base;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_finish(const uint32_t* __restrict__ in, int64_t n,
                                                              const unsigned long long* __restrict__ sums,
                                                              uint64_t* __restrict__ out) {
    // thread owns SCAN_ITEMS consecutive items
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t x[SCAN_ITEMS];
    unsigned long long v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { x[k] = (base + k < n) ? in[base + k] : 0u; v += x[k]; }
    unsigned long long tot;
    unsigned long long run = sums[blockIdx.x] + block_exclusive_scan(v, &tot);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = run;
        run += x[k];
    }
}

int launch_scan_u32(pct_ctx* ctx, const uint32_t* in, uint64_t* out, int64_t n, uint64_t base,
                    unsigned long long* d_total, cudaStream_t st) {
    if (n <= 0) {
        if (d_total) PCT_CUDA(ctx, cudaMemsetAsync(d_total, 0, sizeof(unsigned long long), st));
        return PCT_OK;
    }
    const int64_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    const int64_t need = nb * (int64_t)sizeof(unsigned long long);
    if (need > ctx->scan_tmp_bytes) {
        if (ctx->scan_tmp) PCT_CUDA(ctx, cudaFree(ctx->scan_tmp));
        ctx->scan_tmp = nullptr; ctx->scan_tmp_bytes = 0;
        PCT_CUDA(ctx, cudaMalloc(&ctx->scan_tmp, (size_t)need));
        ctx->scan_tmp_bytes = need;
    }
    unsigned long long* sums = (unsigned long long*)ctx->scan_tmp;
    k_scan_tile_sums<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(in, n, sums);
    k_scan_sums<<<1, SCAN_THREADS, 0, st>>>(sums, nb, base, d_total);
    k_scan_finish<<<(unsigned)nb, SCAN_THREADS, 0, st>>>(in, n, sums, out);
    ctx->launches += 3;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

// ---- decode (parity / debug): one thread per history expands its codes to voxel indices -------------------------
__global__ void __launch_bounds__(128) k_decode(const __grid_constant__ DevCfg g, const uint32_t* __restrict__ N,
                                                const int32_t* __restrict__ start, const uint64_t* __restrict__ code_off,
                                                const ulonglong2* __restrict__ codes, int64_t i0, int64_t i1,
                                                const uint64_t* __restrict__ row_ptr, int32_t* __restrict__ voxels) {
    const int64_t i = i0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= i1) return;
    const uint32_t n = N[i];
    if (n == 0) return;
    int32_t* out = voxels + row_ptr[i - i0];
    int32_t v = start[i];
    out[0] = v;
    const ulonglong2* cp = codes + code_off[i];
    for (uint32_t k = 1; k < n; ++k) {
        const uint32_t ci = k - 1, w = ci % CODES_PER_CHUNK;
        const ulonglong2 ch = cp[ci / CODES_PER_CHUNK];
        const unsigned long long word = w < CODES_PER_WORD ? ch.x : ch.y;
        const int code = (int)((word >> (3 * (w % CODES_PER_WORD))) & 7ull);
        const int axis = code >> 1;
        const int mag = axis == 0 ? g.sx : (axis == 1 ? g.sy : g.sz);
        v += (code & 1) ? -mag : mag;
        out[k] = v;
    }
}

// ---- indices of the histories whose flags intersect `mask` (the tie log, R9) ------------------------------------------
__global__ void __launch_bounds__(256) k_collect_flagged(const uint8_t* __restrict__ flags, int64_t m, unsigned mask,
                                                         uint32_t* __restrict__ idx, int64_t cap, unsigned long long* __restrict__ count) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += stride) {
        if (flags[i] & mask) {
            const unsigned long long slot = atomicAdd(count, 1ull);
            if ((int64_t)slot < cap) idx[slot] = (uint32_t)i;
        }
    }
}

int launch_collect_flagged(pct_ctx* ctx, const pct_paths* P, unsigned mask, uint32_t* idx, int64_t cap, unsigned long long* d_count, cudaStream_t st) {
    PCT_CUDA(ctx, cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), st));
    const int64_t want = (P->m + 255) / 256, lim = (int64_t)ctx->num_sms * 16;
    k_collect_flagged<<<(unsigned)(want < lim ? want : lim), 256, 0, st>>>(P->flags, P->m, mask, idx, cap, d_count);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

int launch_decode(pct_ctx* ctx, const pct_paths* P, int64_t i0, int64_t i1, const uint64_t* row_ptr, int32_t* voxels,
                  cudaStream_t st) {
    const int64_t cnt = i1 - i0;
    if (cnt <= 0) return PCT_OK;
    k_decode<<<(unsigned)((cnt + 127) / 128), 128, 0, st>>>(ctx->cfg, P->N, P->start, P->code_off, P->codes, i0, i1,
                                                            row_ptr, voxels);
    ++ctx->launches;
    PCT_CUDA(ctx, cudaGetLastError());
    return PCT_OK;
}

}  // namespace pct
