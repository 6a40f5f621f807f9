// pcto.cpp -- CPU ORACLE for the pCT hot path of arxiv 1802.01070.  TEST INFRASTRUCTURE ONLY.
//
// Plain FP64 C++17, written for checking by eye against PAPER.md (:7 model and MLP, :98 DROP) and the
// readings R1..R20 of DESIGN.md.  No blocking, fusion or reordering beyond what those state.  OpenMP is
// used only as an outer "parallel for" over independent histories.  Shares nothing with the CUDA path.
//
// Parity status: the paper prints no worked value, so "parity with the paper's numbers" is UNPINNED for
// every function here; each function is instead pinned by the mathematics (tests/test_oracle_*.py):
//   scatter_moments  vs adaptive quadrature (scipy)              mlp_point  vs cubic Hermite spline,
//   straight-line identity, end-point limits, scale invariance, an independent algebraic form
//   hull entry + walk  vs Siddon's exact ray tracing and brute-force dense sampling of the polyline
//   solve  vs dense-matrix DROP / Kaczmarz / least squares in numpy.
#include "pcto.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------------------------------------
// R1: frames.  Grid frame (x,y,z), z = rotation axis; gantry frame (u,t,v), u = beam, v = z.
// ------------------------------------------------------------------------------------------------
struct Grid {
    int n[3];
    double h, lo[3], hi[3];
    explicit Grid(const pcto_geometry& g) {
        n[0] = g.nx; n[1] = g.ny; n[2] = g.nz;
        h = g.h_mm;
        for (int a = 0; a < 3; ++a) { lo[a] = g.origin_mm[a]; hi[a] = g.origin_mm[a] + n[a] * g.h_mm; }
    }
    double face(int a, int i) const { return lo[a] + i * h; }   // plane between voxels i-1 and i on axis a
    bool inside(const int c[3]) const {
        return c[0] >= 0 && c[0] < n[0] && c[1] >= 0 && c[1] < n[1] && c[2] >= 0 && c[2] < n[2];
    }
    int32_t linear(const int c[3]) const { return c[0] + n[0] * (c[1] + n[1] * c[2]); }
    void unlinear(int32_t j, int c[3]) const { c[0] = j % n[0]; c[1] = (j / n[0]) % n[1]; c[2] = j / (n[0] * n[1]); }
};

void gantry_to_grid(double cph, double sph, double u, double t, double v, double p[3]) {
    p[0] = u * cph - t * sph;
    p[1] = u * sph + t * cph;
    p[2] = v;
}
void grid_to_gantry(double cph, double sph, const double p[3], double* u, double* t, double* v) {
    *u = p[0] * cph + p[1] * sph;
    *t = -p[0] * sph + p[1] * cph;
    *v = p[2];
}
double dist3(const double a[3], const double b[3]) {
    const double dx = b[0] - a[0], dy = b[1] - a[1], dz = b[2] - a[2];
    return std::sqrt(dx * dx + dy * dy + dz * dz);
}

// ------------------------------------------------------------------------------------------------
// R9: closed-voxel lazy stepping.  c is the current voxel, A->B the current segment.  If B lies in the
// closed box of c nothing happens.  Otherwise, among the axes on which B is STRICTLY outside, cross the
// face (in the direction of travel) with the smallest segment parameter s; exact equality -> lowest axis.
// A runner-up within tie_eps (measured in mm along the segment) is reported as a tie.
// ------------------------------------------------------------------------------------------------
enum StepResult { STEP_NONE, STEP_OK, STEP_LEFT_GRID };
struct StepInfo { int axis, dir; double s; bool tie; };

StepResult lazy_step(const Grid& g, const double A[3], const double B[3], double seg_len, double tie_eps,
                     int c[3], StepInfo* info) {
    double s[3] = {0, 0, 0};
    int dir[3] = {0, 0, 0};
    for (int a = 0; a < 3; ++a) {
        const double f_lo = g.face(a, c[a]), f_hi = g.face(a, c[a] + 1);
        if (B[a] > f_hi) { dir[a] = +1; s[a] = (f_hi - A[a]) / (B[a] - A[a]); }
        else if (B[a] < f_lo) { dir[a] = -1; s[a] = (f_lo - A[a]) / (B[a] - A[a]); }
    }
    int best = -1;
    for (int a = 0; a < 3; ++a)
        if (dir[a] != 0 && (best < 0 || s[a] < s[best])) best = a;
    if (best < 0) return STEP_NONE;
    bool tie = false;
    for (int a = 0; a < 3; ++a)
        if (a != best && dir[a] != 0 && (s[a] - s[best]) * seg_len < tie_eps) tie = true;
    c[best] += dir[best];
    info->axis = best; info->dir = dir[best]; info->s = s[best]; info->tie = tie;
    return g.inside(c) ? STEP_OK : STEP_LEFT_GRID;
}

// ------------------------------------------------------------------------------------------------
// A1 / R3-R4: from tracker point T along direction d (not normalised) to the first hull voxel.
// ------------------------------------------------------------------------------------------------
struct HullHit { bool ok; bool tie; int c[3]; double P[3]; };

HullHit find_hull(const Grid& g, const uint8_t* hull, const double T[3], const double d[3], double tie_eps) {
    HullHit hit; hit.ok = false; hit.tie = false;
    const double INF = std::numeric_limits<double>::infinity();
    // slab clipping of the ray {T + s d, s >= 0} against the grid box
    double s_min = 0.0, s_max = INF, near_s[3] = {-INF, -INF, -INF};
    int enter_axis = -1;
    for (int a = 0; a < 3; ++a) {
        if (d[a] != 0.0) {
            const double s1 = (g.lo[a] - T[a]) / d[a], s2 = (g.hi[a] - T[a]) / d[a];
            near_s[a] = std::min(s1, s2);
            if (near_s[a] > s_min) { s_min = near_s[a]; enter_axis = a; }
            s_max = std::min(s_max, std::max(s1, s2));
        } else if (T[a] < g.lo[a] || T[a] > g.hi[a]) return hit;
    }
    if (!(s_min < s_max)) return hit;
    const double d_len = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double A[3], B[3];
    for (int a = 0; a < 3; ++a) { A[a] = T[a] + s_min * d[a]; B[a] = T[a] + s_max * d[a]; }
    int c[3];
    for (int a = 0; a < 3; ++a) {
        if (a == enter_axis) {                       // enters through this face: boundary index, exact coordinate
            A[a] = d[a] > 0 ? g.lo[a] : g.hi[a];
            c[a] = d[a] > 0 ? 0 : g.n[a] - 1;
        } else {
            if (enter_axis >= 0 && (s_min - near_s[a]) * d_len < tie_eps) hit.tie = true;   // through a box edge
            const int i = (int)std::floor((A[a] - g.lo[a]) / g.h);
            c[a] = std::min(std::max(i, 0), g.n[a] - 1);
        }
    }
    // walk the chord A->B with rule R9 until the first hull voxel
    const double seg_len = dist3(A, B);
    StepInfo last; last.axis = -1; last.dir = 0; last.s = 0; last.tie = false;
    while (hull != nullptr && hull[g.linear(c)] == 0) {
        StepInfo info;
        if (lazy_step(g, A, B, seg_len, tie_eps, c, &info) != STEP_OK) return hit;   // chord ended or left the grid
        if (info.tie) hit.tie = true;
        last = info;
    }
    for (int a = 0; a < 3; ++a) { hit.c[a] = c[a]; hit.P[a] = last.axis < 0 ? A[a] : A[a] + last.s * (B[a] - A[a]); }
    if (last.axis >= 0)      // the coordinate on the crossed axis is the face itself, exactly
        hit.P[last.axis] = last.dir > 0 ? g.face(last.axis, c[last.axis]) : g.face(last.axis, c[last.axis] + 1);
    hit.ok = true;
    return hit;
}

// ------------------------------------------------------------------------------------------------
// A2 / R6-R7: scattering moments and the MLP of ref [3]
// ------------------------------------------------------------------------------------------------
// { int_{w_a}^{w_b} (W-w)^q f(w) dw, q = 2,1,0 },  f(w) = sum_i a_i w^i.
// Exact polynomial integration in the lever-arm variable r = W - w (no W^2*M0 - 2W*M1 + M2 cancellation):
// f(W - r) = sum_j c_j r^j with c_j = (-1)^j sum_{i>=j} a_i binom(i,j) W^(i-j).
double ipow(double x, int e) { double r = 1.0; for (int k = 0; k < e; ++k) r *= x; return r; }

void scatter_moments(const double a[6], double w_a, double w_b, double W, double out[3]) {
    static const double binom[6][6] = {{1, 0, 0, 0, 0, 0}, {1, 1, 0, 0, 0, 0}, {1, 2, 1, 0, 0, 0},
                                       {1, 3, 3, 1, 0, 0}, {1, 4, 6, 4, 1, 0}, {1, 5, 10, 10, 5, 1}};
    double c[6];
    for (int j = 0; j < 6; ++j) {
        double sum = 0.0;
        for (int i = j; i < 6; ++i) sum += a[i] * binom[i][j] * ipow(W, i - j);
        c[j] = (j % 2 == 0) ? sum : -sum;
    }
    const double r_lo = W - w_b, r_hi = W - w_a;
    for (int q = 0; q <= 2; ++q) {
        double sum = 0.0;
        for (int j = 0; j < 6; ++j) {
            const int e = j + q + 1;
            sum += c[j] * (ipow(r_hi, e) - ipow(r_lo, e)) / e;
        }
        out[2 - q] = sum;
    }
}

struct Mat2 { double a, b, c, d; };   // [[a,b],[c,d]]
Mat2 mul(const Mat2& p, const Mat2& q) {
    return {p.a * q.a + p.b * q.c, p.a * q.b + p.b * q.d, p.c * q.a + p.d * q.c, p.c * q.b + p.d * q.d};
}
Mat2 add(const Mat2& p, const Mat2& q) { return {p.a + q.a, p.b + q.b, p.c + q.c, p.d + q.d}; }
Mat2 transpose(const Mat2& p) { return {p.a, p.c, p.b, p.d}; }
Mat2 inverse(const Mat2& p) {
    const double det = p.a * p.d - p.b * p.c;
    return {p.d / det, -p.b / det, -p.c / det, p.a / det};
}
void mulv(const Mat2& p, const double x[2], double y[2]) { y[0] = p.a * x[0] + p.b * x[1]; y[1] = p.c * x[0] + p.d * x[1]; }

// y_MLP(u1) = (S1^-1 + R1^T S2^-1 R1)^-1 (S1^-1 R0 y0 + R1^T S2^-1 y2), depth w1 = u1-u0 in (0, D), D = u2-u0.
void mlp_point(const pcto_mlp_params& p, double D, double w1, const double y0[2], const double y2[2], double y[2]) {
    const double E0 = 13.6;
    const double d1 = w1, d2 = D - w1;
    double m1[3], m2[3];
    scatter_moments(p.poly, 0.0, w1, w1, m1);     // Sigma1: scattering in [u0,u1] seen at u1
    scatter_moments(p.poly, w1, D, D, m2);        // Sigma2: scattering in [u1,u2] seen at u2
    const double l1 = 1.0 + p.log_coeff * std::log(d1 / p.X0_mm), l2 = 1.0 + p.log_coeff * std::log(d2 / p.X0_mm);
    const double g1 = E0 * E0 * l1 * l1 / p.X0_mm, g2 = E0 * E0 * l2 * l2 / p.X0_mm;
    const Mat2 S1 = {g1 * m1[0], g1 * m1[1], g1 * m1[1], g1 * m1[2]};
    const Mat2 S2 = {g2 * m2[0], g2 * m2[1], g2 * m2[1], g2 * m2[2]};
    const Mat2 R0 = {1.0, d1, 0.0, 1.0}, R1 = {1.0, d2, 0.0, 1.0};
    const Mat2 S1i = inverse(S1), S2i = inverse(S2), R1t = transpose(R1);
    const Mat2 P = add(S1i, mul(R1t, mul(S2i, R1)));
    double r0y0[2], lhs[2], s2y2[2], rhs2[2], rhs[2];
    mulv(R0, y0, r0y0);
    mulv(S1i, r0y0, lhs);
    mulv(S2i, y2, s2y2);
    mulv(R1t, s2y2, rhs2);
    rhs[0] = lhs[0] + rhs2[0];
    rhs[1] = lhs[1] + rhs2[1];
    mulv(inverse(P), rhs, y);
}

// ------------------------------------------------------------------------------------------------
// A1-A3 for one history
// ------------------------------------------------------------------------------------------------
struct Row {
    uint8_t flags = 0;
    double length = 0.0;
    int v_start = -1, v_end = -1;
    std::vector<int32_t> voxels;
    std::vector<double> verts;   // only filled when keep_verts
};

// R9 walk over a polyline; c starts as the start voxel (never from floor() of a point on a face).
// returns false if the walk left the grid.
bool walk_polyline(const Grid& g, double tie_eps, const double* verts, int nverts, int c[3],
                   std::vector<int32_t>* voxels, double* length, int* n_ties) {
    voxels->push_back(g.linear(c));
    for (int k = 0; k + 1 < nverts; ++k) {
        const double* A = verts + 3 * k;
        const double* B = verts + 3 * (k + 1);
        const double seg_len = dist3(A, B);
        *length += seg_len;
        for (;;) {
            StepInfo info;
            const StepResult r = lazy_step(g, A, B, seg_len, tie_eps, c, &info);
            if (r == STEP_NONE) break;
            if (r == STEP_LEFT_GRID) return false;
            if (info.tie) ++*n_ties;
            voxels->push_back(g.linear(c));
        }
    }
    return true;
}

void compute_row(const Grid& g, const pcto_mlp_params& p, const pcto_protons& pr, int64_t i, const uint8_t* hull,
                 bool keep_verts, Row* row) {
    row->flags = 0; row->length = 0.0; row->voxels.clear(); row->verts.clear();
    const double in[9] = {pr.phi[i], pr.t_in[i], pr.v_in[i], pr.dt_in[i], pr.dv_in[i],
                          pr.t_out[i], pr.v_out[i], pr.dt_out[i], pr.dv_out[i]};
    for (double x : in) if (!std::isfinite(x)) { row->flags = PCTO_REJ_NONFINITE; return; }
    const double cph = std::cos(in[0]), sph = std::sin(in[0]);
    // R4: entry ray from the front tracker, exit ray (reversed) from the rear tracker
    double T_in[3], d_in[3], T_out[3], d_out[3];
    gantry_to_grid(cph, sph, pr.u_in_mm, in[1], in[2], T_in);
    gantry_to_grid(cph, sph, 1.0, in[3], in[4], d_in);
    gantry_to_grid(cph, sph, pr.u_out_mm, in[5], in[6], T_out);
    gantry_to_grid(cph, sph, 1.0, in[7], in[8], d_out);
    for (int a = 0; a < 3; ++a) d_out[a] = -d_out[a];
    const HullHit h_in = find_hull(g, hull, T_in, d_in, p.tie_eps_mm);
    const HullHit h_out = find_hull(g, hull, T_out, d_out, p.tie_eps_mm);
    if (!h_in.ok || !h_out.ok) { row->flags = PCTO_REJ_MISS; return; }
    if (h_in.tie || h_out.tie) row->flags |= PCTO_TIE;
    // R5: MLP end states in the gantry frame; slopes are the tracker slopes (straight flight in air)
    double u0, t0, v0, u2, t2, v2;
    grid_to_gantry(cph, sph, h_in.P, &u0, &t0, &v0);
    grid_to_gantry(cph, sph, h_out.P, &u2, &t2, &v2);
    const double D = u2 - u0;
    if (!(D > 0.0)) { row->flags = PCTO_REJ_ORDER; return; }
    if (D > p.poly_max_depth_mm) { row->flags = PCTO_REJ_DEPTH; return; }
    // R8: K uniform steps; the 1e-9 moves the ceil() decision off exact multiples of the nominal step
    const int K = std::max(1, (int)std::ceil(D / (p.step_frac * g.h) - 1e-9));
    const double du = D / K;
    std::vector<double> verts(3 * (size_t)(K + 1));
    for (int a = 0; a < 3; ++a) { verts[a] = h_in.P[a]; verts[3 * (size_t)K + a] = h_out.P[a]; }
    const double yt0[2] = {t0, in[3]}, yt2[2] = {t2, in[7]}, yv0[2] = {v0, in[4]}, yv2[2] = {v2, in[8]};
    for (int k = 1; k < K; ++k) {
        const double w1 = k * du;
        double yt[2], yv[2];
        mlp_point(p, D, w1, yt0, yt2, yt);
        mlp_point(p, D, w1, yv0, yv2, yv);
        gantry_to_grid(cph, sph, u0 + w1, yt[0], yv[0], &verts[3 * (size_t)k]);
    }
    // R9-R11: visit list
    int c[3] = {h_in.c[0], h_in.c[1], h_in.c[2]};
    int n_ties = 0;
    row->v_start = g.linear(h_in.c);
    row->v_end = g.linear(h_out.c);
    const bool ok = walk_polyline(g, p.tie_eps_mm, verts.data(), K + 1, c, &row->voxels, &row->length, &n_ties);
    if (keep_verts) row->verts = verts;
    if (!ok) { row->flags = PCTO_REJ_LEFT_GRID; row->voxels.clear(); return; }
    if ((int64_t)row->voxels.size() > p.max_visits) { row->flags = PCTO_REJ_CAPACITY; row->voxels.clear(); return; }
    if (n_ties > 0) row->flags |= PCTO_TIE;
    if (g.linear(c) != row->v_end) row->flags |= PCTO_END_MISMATCH;   // R10
}

int resolve_threads(int nthreads) {
#ifdef _OPENMP
    return nthreads > 0 ? nthreads : omp_get_max_threads();
#else
    (void)nthreads; return 1;
#endif
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// visit lists of all histories: CSR in chunks (each chunk built by one thread)
// ------------------------------------------------------------------------------------------------
struct pcto_paths {
    static const int64_t CH = 8192;
    int64_t m = 0, n_vox = 0, total_visits = 0, n_rejected = 0, n_ties = 0;
    struct Chunk { std::vector<int64_t> ptr; std::vector<int32_t> vox; };
    std::vector<Chunk> chunks;
    std::vector<float> ell;
    std::vector<uint8_t> flags;
    std::vector<double> length;
    const int32_t* row(int64_t i, int64_t* n) const {
        const Chunk& ch = chunks[i / CH];
        const int64_t k = i % CH;
        *n = ch.ptr[k + 1] - ch.ptr[k];
        return ch.vox.data() + ch.ptr[k];
    }
};

extern "C" {

pcto_paths* pcto_generate_mlp(const pcto_geometry* geom, const pcto_mlp_params* params, const pcto_protons* pr,
                              const uint8_t* hull, int nthreads) {
    if (!geom || !params || !pr || pr->m < 0 || geom->nx <= 0 || geom->ny <= 0 || geom->nz <= 0 ||
        !(geom->h_mm > 0) || !(params->step_frac > 0) || params->max_visits < 1) return nullptr;
    const Grid g(*geom);
    pcto_paths* P = new pcto_paths;
    P->m = pr->m;
    P->n_vox = (int64_t)geom->nx * geom->ny * geom->nz;
    P->ell.assign(pr->m, 0.f);
    P->flags.assign(pr->m, 0);
    P->length.assign(pr->m, 0.0);
    const int64_t nch = (pr->m + pcto_paths::CH - 1) / pcto_paths::CH;
    P->chunks.resize(nch);
    const int nt = resolve_threads(nthreads);
    (void)nt;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
    for (int64_t ci = 0; ci < nch; ++ci) {
        pcto_paths::Chunk& ch = P->chunks[ci];
        const int64_t i0 = ci * pcto_paths::CH, i1 = std::min(pr->m, i0 + pcto_paths::CH);
        ch.ptr.assign(i1 - i0 + 1, 0);
        Row row;
        for (int64_t i = i0; i < i1; ++i) {
            compute_row(g, *params, *pr, i, hull, false, &row);
            const int64_t N = (int64_t)row.voxels.size();
            ch.vox.insert(ch.vox.end(), row.voxels.begin(), row.voxels.end());
            ch.ptr[i - i0 + 1] = ch.ptr[i - i0] + N;
            P->flags[i] = row.flags;
            P->length[i] = N > 0 ? row.length : 0.0;
            P->ell[i] = N > 0 ? (float)(row.length / (double)N) : 0.f;   // R11: mean chord
        }
    }
    for (int64_t ci = 0; ci < nch; ++ci) P->total_visits += (int64_t)P->chunks[ci].vox.size();
    for (int64_t i = 0; i < pr->m; ++i) {
        int64_t N; P->row(i, &N);
        if (N == 0) ++P->n_rejected;
        if (P->flags[i] & PCTO_TIE) ++P->n_ties;
    }
    return P;
}

int pcto_paths_info(const pcto_paths* P, int64_t* m, int64_t* total_visits, int64_t* n_rejected, int64_t* n_ties) {
    if (!P) return -1;
    if (m) *m = P->m;
    if (total_visits) *total_visits = P->total_visits;
    if (n_rejected) *n_rejected = P->n_rejected;
    if (n_ties) *n_ties = P->n_ties;
    return 0;
}

int pcto_paths_rows(const pcto_paths* P, int64_t i0, int64_t i1, int64_t* row_ptr, int32_t* voxels, int64_t cap,
                    float* ell, uint8_t* flags, double* length_mm) {
    if (!P || i0 < 0 || i1 > P->m || i0 > i1 || !row_ptr) return -1;
    int64_t pos = 0;
    row_ptr[0] = 0;
    for (int64_t i = i0; i < i1; ++i) {
        int64_t N; const int32_t* r = P->row(i, &N);
        if (voxels) {
            if (pos + N > cap) return -2;
            std::memcpy(voxels + pos, r, sizeof(int32_t) * (size_t)N);
        }
        pos += N;
        row_ptr[i - i0 + 1] = pos;
        if (ell) ell[i - i0] = P->ell[i];
        if (flags) flags[i - i0] = P->flags[i];
        if (length_mm) length_mm[i - i0] = P->length[i];
    }
    return 0;
}

void pcto_paths_free(pcto_paths* P) { delete P; }

// R19: b_i = l_i * sum over visits of x_j
int pcto_forward_project(const pcto_paths* P, const float* x, float* b_out, int nthreads) {
    if (!P || !x || !b_out) return -1;
    const int nt = resolve_threads(nthreads);
    (void)nt;
#pragma omp parallel for schedule(static) num_threads(nt)
    for (int64_t i = 0; i < P->m; ++i) {
        int64_t N; const int32_t* r = P->row(i, &N);
        double S = 0.0;
        for (int64_t k = 0; k < N; ++k) S += (double)x[r[k]];
        b_out[i] = (float)((double)P->ell[i] * S);
    }
    return 0;
}

// R20: counts_j = number of visits of voxel j by histories [i0,i1)
int pcto_column_counts(const pcto_paths* P, int64_t i0, int64_t i1, uint32_t* counts) {
    if (!P || !counts || i0 < 0 || i1 > P->m || i0 > i1) return -1;
    std::fill(counts, counts + P->n_vox, 0u);
    for (int64_t i = i0; i < i1; ++i) {
        int64_t N; const int32_t* r = P->row(i, &N);
        for (int64_t k = 0; k < N; ++k) ++counts[r[k]];
    }
    return 0;
}

// R13-R18: DROP with unit weights (ref [11]):
//   x <- x + lambda * U_t * sum_{i in B_t} [(b_i - <a_i,x>) / ||a_i||^2] a_i,   U_t = diag(1/max(1,s_j^t)),
//   a_i = l_i on every visit (R12), ||a_i||^2 = N_i l_i^2, so each visit receives c_i = (b_i - l_i S_i)/(N_i l_i).
int pcto_solve(const pcto_paths* P, const float* b, const float* x0, int iters, int64_t block_size, double lambda,
               float* x_out, double* x_out_f64, int nthreads) {
    if (!P || !b || !x0 || iters < 0 || block_size < 1 || (!x_out && !x_out_f64)) return -1;
    const int64_t n = P->n_vox, m = P->m;
    std::vector<double> x(x0, x0 + n), delta(n, 0.0), c((size_t)std::min(block_size, std::max<int64_t>(m, 1)));
    std::vector<uint32_t> s(n, 0u);
    std::vector<int32_t> touched;
    const int nt = resolve_threads(nthreads);
    (void)nt;
    for (int it = 0; it < iters; ++it) {
        for (int64_t i0 = 0; i0 < m; i0 += block_size) {            // R13: consecutive blocks, short tail
            const int64_t i1 = std::min(m, i0 + block_size);
            // R14: all residuals of the block use x as it was at the start of the block
#pragma omp parallel for schedule(static) num_threads(nt)
            for (int64_t i = i0; i < i1; ++i) {
                int64_t N; const int32_t* r = P->row(i, &N);
                double S = 0.0;
                for (int64_t k = 0; k < N; ++k) S += x[r[k]];
                const double l = (double)P->ell[i];
                c[i - i0] = N > 0 ? ((double)b[i] - l * S) / ((double)N * l) : 0.0;   // R17
            }
            for (int64_t i = i0; i < i1; ++i) {                      // R15: s counts visits
                int64_t N; const int32_t* r = P->row(i, &N);
                for (int64_t k = 0; k < N; ++k) {
                    const int32_t j = r[k];
                    if (s[j]++ == 0) touched.push_back(j);
                    delta[j] += c[i - i0];
                }
            }
            for (int32_t j : touched) {                              // R16: constant lambda, no clamp
                x[j] += lambda * delta[j] / (double)std::max<uint32_t>(1u, s[j]);
                delta[j] = 0.0; s[j] = 0u;
            }
            touched.clear();
        }
    }
    for (int64_t j = 0; j < n; ++j) {
        if (x_out) x_out[j] = (float)x[j];
        if (x_out_f64) x_out_f64[j] = x[j];
    }
    return 0;
}

// R27: the same iteration with per-history weights and a box clamp (ref [9]-style options, "standard
// iterative solver [9]"):  x <- clamp( x + lambda * U_t * sum_{i in B_t} w_i [(b_i - <a_i,x>) / ||a_i||^2] a_i ),
// U_t as in pcto_solve (visit counts, independent of w), the clamp applied to the voxels the block touched.
int pcto_solve_ex(const pcto_paths* P, const float* b, const float* x0, const float* w, int iters, int64_t block_size,
                  double lambda, double clamp_lo, double clamp_hi, float* x_out, double* x_out_f64, int nthreads) {
    if (!P || !b || !x0 || iters < 0 || block_size < 1 || (!x_out && !x_out_f64)) return -1;
    (void)nthreads;
    const int64_t n = P->n_vox, m = P->m;
    const bool clamp = clamp_lo <= clamp_hi;
    std::vector<double> x(x0, x0 + n), delta(n, 0.0);
    std::vector<uint32_t> s(n, 0u);
    std::vector<int32_t> touched;
    std::vector<double> c((size_t)std::min(block_size, std::max<int64_t>(m, 1)));
    for (int it = 0; it < iters; ++it) {
        for (int64_t i0 = 0; i0 < m; i0 += block_size) {
            const int64_t i1 = std::min(m, i0 + block_size);
            for (int64_t i = i0; i < i1; ++i) {                       // R14: residuals against the x of the block's start
                int64_t N; const int32_t* r = P->row(i, &N);
                double S = 0.0;
                for (int64_t k = 0; k < N; ++k) S += x[r[k]];
                const double l = (double)P->ell[i], wi = w ? (double)w[i] : 1.0;
                c[i - i0] = N > 0 ? wi * ((double)b[i] - l * S) / ((double)N * l) : 0.0;
            }
            for (int64_t i = i0; i < i1; ++i) {
                int64_t N; const int32_t* r = P->row(i, &N);
                for (int64_t k = 0; k < N; ++k) {
                    const int32_t j = r[k];
                    if (s[j]++ == 0) touched.push_back(j);
                    delta[j] += c[i - i0];
                }
            }
            for (int32_t j : touched) {
                x[j] += lambda * delta[j] / (double)std::max<uint32_t>(1u, s[j]);
                if (clamp) x[j] = std::min(std::max(x[j], clamp_lo), clamp_hi);
                delta[j] = 0.0; s[j] = 0u;
            }
            touched.clear();
        }
    }
    for (int64_t j = 0; j < n; ++j) {
        if (x_out) x_out[j] = (float)x[j];
        if (x_out_f64) x_out_f64[j] = x[j];
    }
    return 0;
}

int pcto_scatter_moments(const pcto_mlp_params* p, double w_a, double w_b, double W, double out[3]) {
    if (!p || !out) return -1;
    scatter_moments(p->poly, w_a, w_b, W, out);
    return 0;
}

int pcto_mlp_point(const pcto_mlp_params* p, double D, double w1, const double y0[2], const double y2[2],
                   double y_out[2]) {
    if (!p || !(w1 > 0.0) || !(w1 < D)) return -1;
    mlp_point(*p, D, w1, y0, y2, y_out);
    return 0;
}

int pcto_polyline(const pcto_geometry* geom, const pcto_mlp_params* params, const pcto_protons* pr, int64_t i,
                  const uint8_t* hull, double* verts_xyz, int cap_verts, int32_t* v_start, int32_t* v_end) {
    if (!geom || !params || !pr || i < 0 || i >= pr->m) return -1;
    const Grid g(*geom);
    Row row;
    compute_row(g, *params, *pr, i, hull, true, &row);
    if (row.verts.empty()) return -2 - (int)row.flags;
    const int nv = (int)(row.verts.size() / 3);
    if (nv > cap_verts) return -1;
    std::memcpy(verts_xyz, row.verts.data(), sizeof(double) * row.verts.size());
    if (v_start) *v_start = row.v_start;
    if (v_end) *v_end = row.v_end;
    return nv;
}

int pcto_walk_polyline(const pcto_geometry* geom, double tie_eps_mm, const double* verts_xyz, int nverts,
                       int32_t start_voxel, int32_t* voxels, int cap, int32_t* n_ties) {
    if (!geom || !verts_xyz || nverts < 1 || !voxels) return -1;
    const Grid g(*geom);
    int c[3];
    g.unlinear(start_voxel, c);
    std::vector<int32_t> list;
    double length = 0.0;
    int ties = 0;
    if (!walk_polyline(g, tie_eps_mm, verts_xyz, nverts, c, &list, &length, &ties)) return -2;
    if ((int)list.size() > cap) return -3;
    std::memcpy(voxels, list.data(), sizeof(int32_t) * list.size());
    if (n_ties) *n_ties = ties;
    return (int)list.size();
}

}  // extern "C"
