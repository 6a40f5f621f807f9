/* pcto.h -- C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, FP64, obviously-correct restatement of the proton-CT hot path of arxiv 1802.01070:
 *   PAPER.md:7   "calculating the individual proton's most likely path [3] ... Ax = b, A containing the
 *                 path data, b the WEPLs, x the relative stopping powers"
 *   PAPER.md:98  "block iterative technique Diagonally-Relaxed Orthogonal Projections (DROP [11])",
 *                 "block size is the number of protons to be processed in parallel"
 * The paper prints no formula; every step below the level of those sentences follows a reading R1..R20
 * listed in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this
 * library.  It shares no code, header, table or helper with the CUDA path under paper_1802_01070_b200/.
 * All pointers are HOST pointers owned by the caller.  Functions return 0 on success, <0 on bad arguments.
 */
#ifndef PCTO_H
#define PCTO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t nx, ny, nz;
    double h_mm;
    double origin_mm[3]; /* lower corner of voxel (0,0,0) in the grid frame (R1) */
} pcto_geometry;

typedef struct {
    double poly[6];           /* f(w) = 1/(beta^2 p^2) = sum a_i w^i, w = depth from hull entry in mm (R6) */
    double poly_max_depth_mm; /* reject histories with u2-u0 beyond this */
    double X0_mm;             /* radiation length, 361 mm for water */
    double log_coeff;         /* 0.038; 0 => pure Fermi-Eyges */
    double step_frac;         /* nominal MLP sampling step = step_frac*h (R8) */
    double tie_eps_mm;        /* 1e-9: decisions closer than this are flagged as ties (R9) */
    int32_t max_visits;       /* histories with more path entries are rejected (capacity of the encoding) */
} pcto_mlp_params;

typedef struct {
    int64_t m;
    const double *phi, *t_in, *v_in, *dt_in, *dv_in, *t_out, *v_out, *dt_out, *dv_out;
    double u_in_mm, u_out_mm; /* tracker plane depths in the gantry frame */
} pcto_protons;

/* per-history flag bits (interface constants, also restated in include/pct.h) */
enum {
    PCTO_REJ_MISS = 0x01, PCTO_REJ_ORDER = 0x02, PCTO_REJ_DEPTH = 0x04, PCTO_REJ_LEFT_GRID = 0x08,
    PCTO_TIE = 0x10, PCTO_END_MISMATCH = 0x20, PCTO_REJ_CAPACITY = 0x40, PCTO_REJ_NONFINITE = 0x80
};

typedef struct pcto_paths pcto_paths;

/* A1-A3: tracker records -> visit lists.  hull: uint8[n] or NULL (= all ones).  nthreads<=0: all cores. */
pcto_paths* pcto_generate_mlp(const pcto_geometry*, const pcto_mlp_params*, const pcto_protons*,
                              const uint8_t* hull, int nthreads);
int pcto_paths_info(const pcto_paths*, int64_t* m, int64_t* total_visits, int64_t* n_rejected, int64_t* n_ties);
/* rows [i0,i1): row_ptr[i1-i0+1], voxels[cap], ell/flags/length[i1-i0] (any of the last three may be NULL) */
int pcto_paths_rows(const pcto_paths*, int64_t i0, int64_t i1, int64_t* row_ptr, int32_t* voxels, int64_t cap,
                    float* ell, uint8_t* flags, double* length_mm);
void pcto_paths_free(pcto_paths*);

/* A9, A4, A5-A8 (R13-R20).  x, b are float32 as on the device; accumulation is FP64 (R18). */
int pcto_forward_project(const pcto_paths*, const float* x, float* b_out, int nthreads);
int pcto_column_counts(const pcto_paths*, int64_t i0, int64_t i1, uint32_t* counts);
int pcto_solve(const pcto_paths*, const float* b, const float* x0, int iters, int64_t block_size, double lambda,
               float* x_out, double* x_out_f64 /* may be NULL */, int nthreads);

/* A5-A8 with the options of ref [9]-style solvers (reading R27): per-history weights w_i in [0, 1] (NULL = all one)
 * multiplying the row's correction, x <- x + lambda U_t sum_i w_i [(b_i - <a_i,x>)/||a_i||^2] a_i, and a box clamp
 * x_j <- min(max(x_j, clamp_lo), clamp_hi) applied to the voxels a block updates, right after its update
 * (clamp_lo > clamp_hi = no clamp).  With w = NULL and no clamp this is pcto_solve. */
int pcto_solve_ex(const pcto_paths*, const float* b, const float* x0, const float* w, int iters, int64_t block_size,
                  double lambda, double clamp_lo, double clamp_hi, float* x_out, double* x_out_f64, int nthreads);

/* --- preprocessing in front of the hot path (pcto_pre.cpp; readings R25, R26) --- */
typedef struct {
    int32_t n_theta;   /* direction bins over [0, 2 pi) */
    int32_t n_s;       /* lateral bins of width ds_mm, centred on the rotation axis */
    double ds_mm;
    int32_t min_count; /* bins with fewer histories count as empty (0) */
} pcto_fbp_params;
/* FBP image from tracker records + WEPL.  sino_mean / sino_filtered: [nz][n_theta][n_s] mean WEPL per bin and
 * its ramp-filtered rows, or NULL. */
int pcto_fbp(const pcto_geometry*, const pcto_protons*, const float* b, const pcto_fbp_params*, double* sino_mean,
             double* sino_filtered, double* x0_out);
/* Hull by space carving: voxels crossed (chord > min_chord_mm) by a history with WEPL < wepl_air_mm become 0, all others 1 */
int pcto_hull_carve(const pcto_geometry*, const pcto_protons*, const float* b, double wepl_air_mm, double min_chord_mm,
                    uint8_t* hull_out);

/* --- building blocks exposed for the pins in tests/ --- */
/* out = { int (W-w)^2 f dw, int (W-w) f dw, int f dw } over [w_a, w_b] */
int pcto_scatter_moments(const pcto_mlp_params*, double w_a, double w_b, double W, double out[3]);
/* MLP state (position, slope) at depth w1 in (0,D) between y0 at depth 0 and y2 at depth D (R7, literal form) */
int pcto_mlp_point(const pcto_mlp_params*, double D, double w1, const double y0[2], const double y2[2],
                   double y_out[2]);
/* polyline vertices (grid frame, xyz triples) of history i; returns #vertices (K+1) or <0 if rejected */
int pcto_polyline(const pcto_geometry*, const pcto_mlp_params*, const pcto_protons*, int64_t i,
                  const uint8_t* hull, double* verts_xyz, int cap_verts, int32_t* v_start, int32_t* v_end);
/* R9 walk of an arbitrary polyline starting in voxel start; returns #entries or <0; ties counted */
int pcto_walk_polyline(const pcto_geometry*, double tie_eps_mm, const double* verts_xyz, int nverts,
                       int32_t start_voxel, int32_t* voxels, int cap, int32_t* n_ties);

#ifdef __cplusplus
}
#endif
#endif
