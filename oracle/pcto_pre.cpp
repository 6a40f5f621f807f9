// pcto_pre.cpp -- CPU ORACLE, part 2: the two preprocessing steps in front of the hot path.  TEST INFRASTRUCTURE ONLY.
//
//   pcto_fbp         the filtered-back-projection image the solver starts from ("Using the FBP image as the
//                    initial iterate, one can iteratively solve the system Ax = b"), reading R25 of DESIGN.md
//   pcto_hull_carve  the object hull from the data themselves (space carving; part of the preprocessing the paper folds
//                    into its totals), reading R26 of DESIGN.md
//
// Plain FP64 C++17, each step written out as R25 / R26 state it; no blocking, no fusion, no FFT.  Shares nothing with the
// CUDA path.  The paper prints no formula for either step, so parity with the paper's numbers is UNPINNED; the functions
// are pinned by mathematics in tests/test_oracle_pre.py:
//   pcto_fbp         the Ram-Lak kernel against its closed-form frequency response |f|; the reconstruction of a uniform disc
//                    against its known value; an independent numpy restatement (np.convolve / np.interp); linearity;
//                    invariance under the rebinning of a diverging beam
//   pcto_hull_carve  Siddon's exact chords (numpy) for which voxels a ray may carve; monotonicity; a convex phantom is
//                    recovered up to the one-voxel rim
#include "pcto.h"

#include <cmath>
#include <cstring>
#include <vector>

namespace {
const double PI = 3.14159265358979323846;
}

extern "C" {

// R25.  Every history is taken as the straight chord between its two tracker hits (gantry frame):
//   alpha = atan2(t_out - t_in, u_out - u_in)                   direction of the chord relative to the beam axis
//   theta = phi + alpha (mod 2 pi)                               its direction in the grid frame
//   s     = t_m cos(alpha) - u_m sin(alpha)                      its signed distance from the rotation axis,
//                                                                (u_m, t_m) = midpoint of the two hits
//   z     = (v_in + v_out) / 2                                   its height, taken as constant (paths barely move in z)
// so a diverging beam is rebinned to parallel projections exactly.  Bins: n_theta equal sectors of [0, 2 pi), n_s bins of
// width ds centred on s = 0, one bin per slice; a bin's value is the mean WEPL of its histories (0 if it has fewer than
// min_count).  Each (slice, theta) row is filtered with the band-limited ramp (Ram-Lak) kernel h(0) = 1 / (4 ds^2),
// h(n) = -1 / (pi^2 n^2 ds^2) for odd n, 0 for even n, by direct convolution, q = ds * (p * h); the image value at a voxel
// centre (x, y) of slice z is (pi / n_theta) * sum over theta bins of q interpolated linearly at
// s = -x sin(theta_c) + y cos(theta_c), theta_c the bin centre (full 2 pi of directions, hence pi / n_theta and not
// 2 pi / n_theta).
int pcto_fbp(const pcto_geometry* g, const pcto_protons* pr, const float* b, const pcto_fbp_params* fp,
             double* sino_mean /* [nz][n_theta][n_s] or NULL */, double* sino_filtered /* same shape or NULL */, double* x0_out /* [n] */) {
    if (!g || !pr || !b || !fp || !x0_out || fp->n_theta < 1 || fp->n_s < 2 || !(fp->ds_mm > 0.0) || g->nx <= 0 || g->ny <= 0 ||
        g->nz <= 0 || !(g->h_mm > 0.0)) return -1;
    const int nt = fp->n_theta, ns = fp->n_s, nz = g->nz;
    const double ds = fp->ds_mm, dth = 2.0 * PI / nt;
    const size_t rows = (size_t)nz * nt, cells = rows * ns;
    std::vector<double> sum(cells, 0.0), q(cells, 0.0);
    std::vector<int64_t> cnt(cells, 0);
    for (int64_t i = 0; i < pr->m; ++i) {
        const double in[8] = {pr->phi[i], pr->t_in[i], pr->v_in[i], pr->t_out[i], pr->v_out[i], (double)b[i], pr->u_in_mm, pr->u_out_mm};
        bool ok = true;
        for (double x : in) ok = ok && std::isfinite(x);
        if (!ok) continue;
        const double alpha = std::atan2(pr->t_out[i] - pr->t_in[i], pr->u_out_mm - pr->u_in_mm);
        double theta = std::fmod(pr->phi[i] + alpha, 2.0 * PI);
        if (theta < 0.0) theta += 2.0 * PI;
        const double t_m = 0.5 * (pr->t_in[i] + pr->t_out[i]), u_m = 0.5 * (pr->u_in_mm + pr->u_out_mm);
        const double s = t_m * std::cos(alpha) - u_m * std::sin(alpha);
        const double z = 0.5 * (pr->v_in[i] + pr->v_out[i]);
        int it = (int)std::floor(theta / dth);
        if (it >= nt) it = nt - 1;                                   // theta == 2 pi - 0
        const double js_f = std::floor(s / ds + 0.5 * ns), iz_f = std::floor((z - g->origin_mm[2]) / g->h_mm);
        if (js_f < 0.0 || js_f >= (double)ns || iz_f < 0.0 || iz_f >= (double)nz) continue;
        const size_t cell = ((size_t)iz_f * nt + (size_t)it) * ns + (size_t)js_f;
        sum[cell] += (double)b[i];
        cnt[cell] += 1;
    }
    const int64_t min_count = fp->min_count > 1 ? fp->min_count : 1;
    for (size_t c = 0; c < cells; ++c) sum[c] = cnt[c] >= min_count ? sum[c] / (double)cnt[c] : 0.0;     // mean WEPL per bin
    if (sino_mean) std::memcpy(sino_mean, sum.data(), sizeof(double) * cells);
    // ramp filter, row by row, direct convolution
    for (size_t r = 0; r < rows; ++r) {
        const double* p = sum.data() + r * ns;
        double* qr = q.data() + r * ns;
        for (int j = 0; j < ns; ++j) {
            double acc = 0.0;
            for (int k = 0; k < ns; ++k) {
                const int n = j - k;
                double h = 0.0;
                if (n == 0) h = 1.0 / (4.0 * ds * ds);
                else if (n % 2 != 0) h = -1.0 / (PI * PI * (double)n * (double)n * ds * ds);
                acc += p[k] * h;
            }
            qr[j] = ds * acc;
        }
    }
    if (sino_filtered) std::memcpy(sino_filtered, q.data(), sizeof(double) * cells);
    // voxel-driven back projection
    for (int iz = 0; iz < nz; ++iz)
        for (int iy = 0; iy < g->ny; ++iy)
            for (int ix = 0; ix < g->nx; ++ix) {
                const double x = g->origin_mm[0] + (ix + 0.5) * g->h_mm, y = g->origin_mm[1] + (iy + 0.5) * g->h_mm;
                double acc = 0.0;
                for (int it = 0; it < nt; ++it) {
                    const double th = (it + 0.5) * dth;
                    const double s = -x * std::sin(th) + y * std::cos(th);
                    const double u = s / ds + 0.5 * ns - 0.5;                  // bin j is centred on (j + 1/2 - n_s / 2) ds
                    const double j0 = std::floor(u), f = u - j0;
                    const double* qr = q.data() + ((size_t)iz * nt + it) * ns;
                    const double q0 = (j0 >= 0.0 && j0 < (double)ns) ? qr[(int)j0] : 0.0;
                    const double q1 = (j0 + 1.0 >= 0.0 && j0 + 1.0 < (double)ns) ? qr[(int)j0 + 1] : 0.0;
                    acc += (1.0 - f) * q0 + f * q1;
                }
                x0_out[(size_t)ix + (size_t)g->nx * ((size_t)iy + (size_t)g->ny * iz)] = (PI / nt) * acc;
            }
    return 0;
}

// R26.  Space carving: a history whose WEPL is below wepl_air_mm saw (almost) no material, so the straight chord between
// its tracker hits ran through air.  Every voxel that such a chord crosses with a chord length of more than min_chord_mm
// is carved (0); what is never carved stays hull (1).  The chord of a voxel is |B - A| (s_exit - s_entry) with the entry /
// exit parameters of the three slab pairs of the voxel (exact Siddon geometry, voxel by voxel).
int pcto_hull_carve(const pcto_geometry* g, const pcto_protons* pr, const float* b, double wepl_air_mm, double min_chord_mm,
                    uint8_t* hull_out /* [n] */) {
    if (!g || !pr || !b || !hull_out || g->nx <= 0 || g->ny <= 0 || g->nz <= 0 || !(g->h_mm > 0.0) || !(min_chord_mm >= 0.0)) return -1;
    const int n[3] = {g->nx, g->ny, g->nz};
    const size_t nvox = (size_t)n[0] * n[1] * n[2];
    std::memset(hull_out, 1, nvox);
    const double INF = HUGE_VAL;
    for (int64_t i = 0; i < pr->m; ++i) {
        if (!(std::isfinite((double)b[i]) && (double)b[i] < wepl_air_mm)) continue;
        const double in[5] = {pr->phi[i], pr->t_in[i], pr->v_in[i], pr->t_out[i], pr->v_out[i]};
        bool ok = true;
        for (double x : in) ok = ok && std::isfinite(x);
        if (!ok) continue;
        const double c = std::cos(pr->phi[i]), s = std::sin(pr->phi[i]);
        const double A[3] = {pr->u_in_mm * c - pr->t_in[i] * s, pr->u_in_mm * s + pr->t_in[i] * c, pr->v_in[i]};      // R1
        const double B[3] = {pr->u_out_mm * c - pr->t_out[i] * s, pr->u_out_mm * s + pr->t_out[i] * c, pr->v_out[i]};
        const double d[3] = {B[0] - A[0], B[1] - A[1], B[2] - A[2]};
        const double len = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (!(len > 0.0)) continue;
        // the chord's parameter range inside the grid box, then the range of voxel indices it can touch on every axis
        double s_lo = 0.0, s_hi = 1.0;
        bool miss = false;
        for (int a = 0; a < 3; ++a) {
            const double lo = g->origin_mm[a], hi = g->origin_mm[a] + n[a] * g->h_mm;
            if (d[a] != 0.0) {
                const double s1 = (lo - A[a]) / d[a], s2 = (hi - A[a]) / d[a];
                s_lo = std::fmax(s_lo, std::fmin(s1, s2));
                s_hi = std::fmin(s_hi, std::fmax(s1, s2));
            } else if (A[a] < lo || A[a] > hi) miss = true;
        }
        if (miss || !(s_lo < s_hi)) continue;
        int i_lo[3], i_hi[3];
        for (int a = 0; a < 3; ++a) {
            const double p0 = A[a] + s_lo * d[a], p1 = A[a] + s_hi * d[a];
            const double f0 = std::floor((std::fmin(p0, p1) - g->origin_mm[a]) / g->h_mm), f1 = std::floor((std::fmax(p0, p1) - g->origin_mm[a]) / g->h_mm);
            i_lo[a] = (int)std::fmax(0.0, f0 - 1.0);
            i_hi[a] = (int)std::fmin((double)(n[a] - 1), f1 + 1.0);
        }
        // march along the axis of largest extent; for every index there, test the few voxels of the other two axes in range
        int am = 0;
        for (int a = 1; a < 3; ++a) if (std::fabs(d[a]) > std::fabs(d[am])) am = a;
        const int a1 = (am + 1) % 3, a2 = (am + 2) % 3;
        for (int im = i_lo[am]; im <= i_hi[am]; ++im) {
            // parameter range of this slab of the marching axis
            const double lo_m = g->origin_mm[am] + im * g->h_mm, hi_m = g->origin_mm[am] + (im + 1) * g->h_mm;
            const double sa = (lo_m - A[am]) / d[am], sb = (hi_m - A[am]) / d[am];
            const double sm0 = std::fmax(s_lo, std::fmin(sa, sb)), sm1 = std::fmin(s_hi, std::fmax(sa, sb));
            if (!(sm0 < sm1)) continue;
            int r_lo[3], r_hi[3];
            for (int a : {a1, a2}) {
                const double p0 = A[a] + sm0 * d[a], p1 = A[a] + sm1 * d[a];
                r_lo[a] = (int)std::fmax((double)i_lo[a], std::floor((std::fmin(p0, p1) - g->origin_mm[a]) / g->h_mm) - 1.0);
                r_hi[a] = (int)std::fmin((double)i_hi[a], std::floor((std::fmax(p0, p1) - g->origin_mm[a]) / g->h_mm) + 1.0);
            }
            for (int i1 = r_lo[a1]; i1 <= r_hi[a1]; ++i1)
                for (int i2 = r_lo[a2]; i2 <= r_hi[a2]; ++i2) {
                    int idx[3];
                    idx[am] = im; idx[a1] = i1; idx[a2] = i2;
                    double e0 = s_lo, e1 = s_hi;                       // entry / exit parameter of this voxel
                    bool out = false;
                    for (int a = 0; a < 3; ++a) {
                        const double lo = g->origin_mm[a] + idx[a] * g->h_mm, hi = g->origin_mm[a] + (idx[a] + 1) * g->h_mm;
                        if (d[a] != 0.0) {
                            const double s1 = (lo - A[a]) / d[a], s2 = (hi - A[a]) / d[a];
                            e0 = std::fmax(e0, std::fmin(s1, s2));
                            e1 = std::fmin(e1, std::fmax(s1, s2));
                        } else if (A[a] < lo || A[a] > hi) out = true;
                    }
                    if (out || !(e1 > e0)) continue;
                    if ((e1 - e0) * len > min_chord_mm)
                        hull_out[(size_t)idx[0] + (size_t)n[0] * ((size_t)idx[1] + (size_t)n[1] * idx[2])] = 0;
                }
        }
        (void)INF;
    }
    return 0;
}

}  // extern "C"
