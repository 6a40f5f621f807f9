/* pct.h -- C-ABI of libpct.so: the single-B200 hot path of proton-CT reconstruction (arxiv 1802.01070).
 *
 *   PAPER.md:7   "calculating the individual proton's most likely path [3] ... large and sparse linear system
 *                 Ax = b ... A is a m x n matrix containing the path data, b is the m x 1 WEPLs vector, and x is
 *                 the n x 1 relative stopping powers (RSP) vector"                      -> pct_generate_mlp
 *   PAPER.md:98  "block iterative technique Diagonally-Relaxed Orthogonal Projections (DROP [11])", "the block
 *                 size is the number of protons to be processed in parallel"            -> pct_solve
 *   PAPER.md:7   b = A x                                                               -> pct_forward_project
 * The paper prints no formula; the exact operations are the readings R1..R20 in DESIGN.md.
 *
 * Conventions
 *   - Plain C, no C++/torch types.  Every pointer is documented as HOST or DEVICE memory; buffers are owned by
 *     the caller and never retained or freed by the library, except the opaque pct_ctx / pct_paths objects,
 *     which the library owns until pct_destroy / pct_paths_free.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Work is enqueued on it; device
 *     results are valid once the caller has synchronised the stream.  Calls that need sizes on the host synchronise
 *     the stream themselves and say so below: pct_generate_mlp, pct_paths_decode, pct_paths_flagged, pct_fbp,
 *     pct_hull_intersect, pct_region_members, pct_reconstruct_regions, the *_host calls, and the FIRST pct_solve /
 *     pct_solve_ex on a (paths, block_size) pair that builds a solve plan.
 *   - Thread safety: a pct_ctx and a pct_paths are each used by one thread at a time.  pct_solve keeps a solve plan
 *     (a solver-shaped copy of the rows) inside the pct_paths it is given -- hence `pct_paths*`, not const -- and the
 *     block counts of that plan inside the context.
 *   - Out-of-range depth is not an error code: a history whose hull chord exceeds poly_max_depth_mm is rejected with
 *     the flag PCT_REJ_DEPTH (SURVEY.md 8(b) listed PCT_E_DEPTH_RANGE; a per-history condition belongs in the flags).
 *   - Device memory: paths, plans and scratch come from a process-wide cache of device blocks that are reused on an exact
 *     size match (rebuilding the same reconstruction costs no allocation); pct_trim_cache releases the idle blocks, and so
 *     does pct_destroy of the last context of a device.  All calls on one context must be issued on one stream at a time (a
 *     reused block relies on stream order).
 *   - Return value: PCT_OK (0) or a negative PCT_E_* code; never throws, never aborts.  pct_last_error(ctx)
 *     gives a human-readable message for the last failure on that context.
 *   - Frames (R1): grid frame (x,y,z), z = rotation axis, voxel (ix,iy,iz) = origin + [i, i+1]*h per axis,
 *     linear index j = ix + nx*(iy + ny*iz).  Gantry frame (u,t,v): x = u cos(phi) - t sin(phi),
 *     y = u sin(phi) + t cos(phi), z = v.  Slopes are dt/du, dv/du (R2).
 *   - Rejected histories (flags & PCT_REJECT_MASK) have N_i = 0 and contribute nothing anywhere.
 */
#ifndef PCT_H
#define PCT_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define PCT_OK 0
#define PCT_E_INVALID_ARG (-1)
#define PCT_E_OOM (-2)
#define PCT_E_CUDA (-3)
#define PCT_E_CAPACITY (-4)

/* per-history flag bits */
#define PCT_REJ_MISS 0x01      /* entry or exit ray misses the grid box / the hull (R4)            */
#define PCT_REJ_ORDER 0x02     /* hull exit not behind hull entry (u2 <= u0)                       */
#define PCT_REJ_DEPTH 0x04     /* u2 - u0 > poly_max_depth_mm (R6)                                 */
#define PCT_REJ_LEFT_GRID 0x08 /* the walk stepped outside the grid (R10)                          */
#define PCT_TIE 0x10           /* some stepping decision was closer than tie_eps_mm (R9); logged   */
#define PCT_END_MISMATCH 0x20  /* walk did not end in the exit hull voxel (R10); list kept         */
#define PCT_REJ_CAPACITY 0x40  /* more than max_visits path entries                                */
#define PCT_REJ_NONFINITE 0x80 /* NaN/Inf tracker record                                           */
#define PCT_REJECT_MASK (PCT_REJ_MISS | PCT_REJ_ORDER | PCT_REJ_DEPTH | PCT_REJ_LEFT_GRID | PCT_REJ_CAPACITY | PCT_REJ_NONFINITE)

typedef struct pct_ctx pct_ctx;     /* opaque: geometry, MLP constants, device scratch            */
typedef struct pct_paths pct_paths; /* opaque: device-resident encoded rows of A (R9-R12)         */

typedef struct {
    int32_t nx, ny, nz;
    double h_mm;
    double origin_mm[3]; /* lower corner of voxel (0,0,0), grid frame */
} pct_geometry;

typedef struct {
    double poly[6];           /* 1/(beta^2 p^2) = sum a_i w^i, w = depth from hull entry in mm (R6)   */
    double poly_max_depth_mm; /* validity range of poly; deeper histories are rejected                 */
    double X0_mm;             /* radiation length (361 mm, water)                                      */
    double log_coeff;         /* 0.038; 0 => pure Fermi-Eyges                                          */
    double step_frac;         /* nominal MLP step = step_frac * h (R8; 0.5)                            */
    double tie_eps_mm;        /* 1e-9 (R9)                                                             */
    int32_t max_visits;       /* capacity of one encoded row, <= 8192                                  */
} pct_mlp_params;

typedef struct {
    int64_t m;
    /* m doubles each: gantry angle [rad]; entry tracker position/slope; exit tracker position/slope.
     * DEVICE pointers for pct_generate_mlp, HOST pointers for pct_reconstruct_host. */
    const double *phi, *t_in, *v_in, *dt_in, *dv_in, *t_out, *v_out, *dt_out, *dv_out;
    double u_in_mm, u_out_mm; /* tracker plane depths in the gantry frame */
} pct_protons;

typedef struct {
    int64_t m, total_visits, n_rejected, n_ties, code_bytes, header_bytes;
    int64_t total_samples; /* sum of K over the accepted histories: MLP segments evaluated (R8); K1's unit of FP64 work */
    int64_t n_general_segments; /* polyline segments that took K1's general stepping loop instead of the loop-free path (longer
                                 * than a voxel on some axis, leaving the grid, row capacity): same result, slower */
} pct_paths_stats;

typedef struct {
    int64_t m, total_visits, n_rejected, n_ties;
    double ms_h2d, ms_mlp, ms_solve, ms_d2h; /* CUDA-event times of the four phases; the H2D copies of the tracker
                                              * arrays run on a copy stream and overlap ms_mlp */
} pct_recon_stats;

/* Create a context on CUDA device `device`.  Validates geometry/params.  HOST pointers. */
int pct_create(const pct_geometry* geom, const pct_mlp_params* params, int device, pct_ctx** out);
void pct_destroy(pct_ctx* ctx);
const char* pct_last_error(const pct_ctx* ctx);

/* A1-A3: tracker records -> most likely path -> visit list, stored as start voxel + 3-bit face
 * step codes.  protons: struct on HOST holding DEVICE arrays.  hull: DEVICE uint8[n], NULL = every voxel is
 * hull.  *out receives a new pct_paths.  Synchronises `stream`. */
int pct_generate_mlp(pct_ctx* ctx, const pct_protons* protons, const uint8_t* hull, void* stream, pct_paths** out);
int pct_paths_info(const pct_paths* paths, pct_paths_stats* out /* HOST */);
void pct_paths_free(pct_paths* paths);

/* Parity/debug: expand rows [i0,i1) to explicit voxel lists.  All outputs DEVICE; any of voxels/ell/flags may
 * be NULL.  row_ptr: int64[i1-i0+1]; voxels: int32[cap] (PCT_E_CAPACITY if cap is too small; row_ptr is
 * still valid then); ell: float32[i1-i0] mean chord l_i; flags: uint8[i1-i0].  Synchronises `stream`. */
int pct_paths_decode(pct_ctx* ctx, const pct_paths* paths, int64_t i0, int64_t i1, int64_t* row_ptr, int32_t* voxels,
                     int64_t cap, float* ell, uint8_t* flags, void* stream);

/* The tie log (R9; north_star: "logged boundary ties"): indices, ascending, of the histories whose flags intersect
 * `mask` (e.g. PCT_TIE).  idx_out: HOST int64[cap] (may be NULL if cap == 0); *n_out (HOST) = how many histories match.
 * If more than cap match, an arbitrary cap of them are returned.  m < 2^32.  Synchronises `stream`. */
int pct_paths_flagged(pct_ctx* ctx, const pct_paths* paths, uint32_t mask, int64_t* idx_out, int64_t cap, int64_t* n_out,
                      void* stream);

/* A9 (R19): b_out[i] = l_i * sum over visits of x[j].  x: DEVICE float32[n]; b_out: DEVICE float32[m]. */
int pct_forward_project(pct_ctx* ctx, const pct_paths* paths, const float* x, float* b_out, void* stream);

/* A4 (R20): counts[j] = visits of voxel j by histories [i0,i1).  counts: DEVICE uint32[n] (overwritten). */
int pct_column_counts(pct_ctx* ctx, const pct_paths* paths, int64_t i0, int64_t i1, uint32_t* counts, void* stream);

/* A5-A8 (R13-R18): `iters` sweeps of block-iterative DROP with unit weights,
 *   x <- x + lambda * diag(1/max(1,s_j^t)) * sum_{i in block t} [(b_i - <a_i,x>)/||a_i||^2] a_i,
 * blocks = consecutive ranges of block_size histories.  b: DEVICE float32[m]; x0, x_out: DEVICE float32[n],
 * x_out may alias x0.  FP32 arithmetic, FP32 atomics (result unique up to summation order).
 * Blocks of at least 32768 histories (pct_solve_config) run through a solve plan that is built on the first call for this
 * (paths, block_size), cached in `paths` and rebuilt when block_size changes; building it synchronises `stream` several
 * times.  Blocks of at most 4096 histories run in one persistent cooperative kernel; sizes in between launch two kernels
 * per block.  No synchronisation otherwise. */
int pct_solve(pct_ctx* ctx, pct_paths* paths, const float* b, const float* x0, int iters, int64_t block_size,
              float lambda, float* x_out, void* stream);

/* A5-A8 with the options of ref [9]-style solvers ("standard iterative solver [9]"; reading R27):
 *   x <- clamp( x + lambda * diag(1/max(1,s_j^t)) * sum_{i in block t} w_i [(b_i - <a_i,x>)/||a_i||^2] a_i )
 * weights: DEVICE float32[m] in [0, 1] or NULL (= all one); the clamp x_j <- min(max(x_j, clamp_lo), clamp_hi) is applied
 * to the voxels a block updates, right after its update; clamp_lo > clamp_hi = no clamp.  opts == NULL = pct_solve. */
typedef struct {
    const float* weights;
    float clamp_lo, clamp_hi;
} pct_solve_opts;
int pct_solve_ex(pct_ctx* ctx, pct_paths* paths, const float* b, const float* x0, int iters, int64_t block_size,
                 float lambda, const pct_solve_opts* opts /* HOST */, float* x_out, void* stream);

/* The FBP image the solver starts from ("Using the FBP image as the initial iterate"; reading R25): every
 * history is taken as the straight chord between its tracker hits and rebinned to parallel projections (direction
 * theta = phi + alpha, signed distance s from the rotation axis, height z = mean of the two hits); bins: n_theta sectors
 * of [0, 2 pi), n_s bins of ds_mm centred on the axis, one per slice; bin value = mean WEPL (0 below min_count histories);
 * rows filtered with the band-limited ramp (Ram-Lak) kernel by direct convolution; voxel-driven back projection with linear
 * interpolation, x0 = (pi / n_theta) * sum over directions.  FP64 inside, float32 out.
 * protons: HOST struct of DEVICE arrays; b: DEVICE float32[m]; x0_out: DEVICE float32[n].  Synchronises `stream` (its
 * sinogram scratch goes back to the buffer cache). */
typedef struct {
    int32_t n_theta, n_s;
    double ds_mm;
    int32_t min_count;
} pct_fbp_params;
int pct_fbp(pct_ctx* ctx, const pct_protons* protons, const float* b, const pct_fbp_params* params /* HOST */, float* x0_out,
            void* stream);

/* pct_fbp WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under stream capture, serving loops,
 * harnesses that forbid it).  Same arguments, same kernels, same result as pct_fbp; the sinogram scratch (20 bytes per bin)
 * is a fixed device array inside the library sized for PCT_FBP_STATIC_MAX_CELLS bins -- 20 MiB that every GPU which loads
 * the library holds until the process exits.  nz * n_theta * n_s > PCT_FBP_STATIC_MAX_CELLS is rejected with
 * PCT_E_CAPACITY (use pct_fbp).  Calls no cudaMalloc / cudaFree and no allocating library routine; enqueues two memsets (the
 * array keeps the last call's contents) and three kernels on `stream` and does NOT synchronise it.  Every call on a device,
 * from any context, shares the one array: calls that overlap on the GPU (different streams without an ordering between
 * them) race and give garbage; calls on one stream, or ordered by events, are safe. */
#define PCT_FBP_STATIC_MAX_CELLS (1u << 20)
int pct_fbp_static(pct_ctx* ctx, const pct_protons* protons, const float* b, const pct_fbp_params* params /* HOST */,
                   float* x0_out, void* stream);

/* The object hull from the data (space carving; preprocessing of PAPER.md:102-104; reading R26): hull_out[j] = 0 for every
 * voxel that the straight chord between the tracker hits of some history with WEPL < wepl_air_mm crosses with a chord
 * length > min_chord_mm, 1 otherwise.  hull_out: DEVICE uint8[n] (overwritten).  Use min_chord_mm > 0: voxels a chord only
 * grazes at a corner are decided by rounding otherwise.  Enqueued on `stream`. */
int pct_hull_carve(pct_ctx* ctx, const pct_protons* protons, const float* b, double wepl_air_mm, double min_chord_mm,
                   uint8_t* hull_out, void* stream);

/* ---- Algorithm 1 of the paper: "multi-GPU based reconstruction" (reading R28 of DESIGN.md) -------------
 *   1: setupImageRegions()  2: identifyProtonsPassingRegions()  3: allocateMemoryForProtonsPerGPU()
 *   4: iterativelySolvePerGPU()  5: selectSlice()
 * The volume is cut along z into n_regions parts of (almost) equal height; region g reconstructs its part plus `ext` slices
 * of each neighbour ("two regions, one containing slices 0-12 and the other containing slices 7-19": nz = 20,
 * n_regions = 2, ext = 3); a history belongs to every region that holds the slice of its hull entry voxel or of its hull exit
 * voxel ("associated with the image region entered to and exited from"); each region is solved on its own histories only, with
 * no exchange between regions ("eliminating the need of data transfers among the GPUs"); the final image takes
 * the slices of each part from that part's region ("slices 0-9 from the first region and 10-19 of the second").  One region
 * per GPU is the paper's use; one GPU may also run several regions in turn. */
typedef struct {
    int32_t z_lo, z_hi;       /* slices [z_lo, z_hi) the region reconstructs                               */
    int32_t keep_lo, keep_hi; /* slices [keep_lo, keep_hi) of the final image that are taken from it      */
} pct_region;
/* Step 1.  Pure host arithmetic, no context: part g = [g nz / G, (g+1) nz / G) (integer division), region = part widened by
 * ext slices on every side that has a neighbour.  out: HOST pct_region[n_regions].  PCT_E_INVALID_ARG unless
 * 1 <= n_regions <= nz and ext >= 0. */
int pct_regions_setup(int32_t nz, int32_t n_regions, int32_t ext, pct_region* out);
/* A1 alone (R4): the hull entry and exit voxel of every history, -1 / -1 for a history rejected there (miss, order, depth,
 * non-finite record) -- what step 2 needs, at a fifth of the cost of pct_generate_mlp, and equal to the first and last
 * voxel of the row pct_generate_mlp would produce.  protons: HOST struct of DEVICE arrays; hull: DEVICE uint8[n] or NULL;
 * v_in, v_out: DEVICE int32[m].  Synchronises `stream`. */
int pct_hull_intersect(pct_ctx* ctx, const pct_protons* protons, const uint8_t* hull, int32_t* v_in, int32_t* v_out, void* stream);
/* Step 2.  idx_out (DEVICE uint32[m], ascending) = the histories with v_in >= 0 whose entry slice or exit slice lies in
 * [region->z_lo, region->z_hi); *count_out (HOST) = how many.  region: HOST.  m < 2^31.  Synchronises `stream`. */
int pct_region_members(pct_ctx* ctx, const int32_t* v_in, const int32_t* v_out, int64_t m, const pct_region* region,
                       uint32_t* idx_out, int64_t* count_out, void* stream);
/* Step 3.  dst arrays [k] = src arrays [idx[k]], b_dst[k] = b_src[idx[k]] for k < count.  src, dst: HOST structs of DEVICE
 * arrays (dst's nine arrays hold at least `count` doubles each and are written; the call sets dst->m and the tracker planes);
 * b_src / b_dst: DEVICE float32, both NULL to skip.  Enqueued on `stream`. */
int pct_gather_histories(pct_ctx* ctx, const pct_protons* src, const float* b_src, const uint32_t* idx, int64_t count,
                         pct_protons* dst, float* b_dst, void* stream);
/* Step 5.  x_final[slices keep_lo..keep_hi) = x_region[the same slices]; both DEVICE float32[n].  Enqueued on `stream`. */
int pct_select_slices(pct_ctx* ctx, const float* x_region, const pct_region* region /* HOST */, float* x_final, void* stream);
/* Steps 1-5 for the regions [region_first, region_first + region_count) on this context's GPU: pct_hull_intersect on all
 * histories, then per region pct_region_members, pct_gather_histories, pct_generate_mlp and pct_solve on the members (x of the
 * whole grid, started from x0 or from ones; only the region's kept slices are used), pct_select_slices into x_out.  Slices
 * kept by other regions are left as they are in x_out: a process per GPU runs its own region and the kept slices are
 * collected afterwards (the only transfer).  members_out: HOST int64[n_regions] or NULL; entries of the regions
 * run here are set.  protons: HOST struct of DEVICE arrays; b: DEVICE float32[m]; hull: DEVICE uint8[n] or NULL; x0: DEVICE
 * float32[n] or NULL; x_out: DEVICE float32[n], must not alias x0.  n_regions <= 1024.  Blocking. */
int pct_reconstruct_regions(pct_ctx* ctx, const pct_protons* protons, const float* b, const uint8_t* hull, const float* x0,
                            int32_t n_regions, int32_t ext, int32_t region_first, int32_t region_count, int iters,
                            int64_t block_size, float lambda, float* x_out, int64_t* members_out, void* stream);

/* The whole hot path on HOST buffers (bench e2e): H2D of the tracker arrays, hull and b; pct_generate_mlp;
 * pct_solve; D2H of x.  protons: HOST struct with HOST arrays; hull_host: uint8[n] or NULL; b_host: float32[m];
 * x0_host: float32[n] or NULL (= all ones); x_out_host: float32[n]; stats may be NULL.  Blocking. */
int pct_reconstruct_host(pct_ctx* ctx, const pct_protons* protons, const uint8_t* hull_host, const float* b_host,
                         const float* x0_host, int iters, int64_t block_size, float lambda, float* x_out_host,
                         pct_recon_stats* stats, void* stream);

/* Releases the idle blocks of the device-buffer cache of ctx's device (synchronises the device). */
int pct_trim_cache(pct_ctx* ctx);

/* Number of kernel launches issued by this context so far (bench.py reports it as gpu_launches). */
int64_t pct_launch_count(const pct_ctx* ctx);

/* How pct_solve runs a block's projection (A4-A6).  mode 0 (default) = automatic: blocks of at least
 * `min_block` histories (<= 0: library default) use the solve plan -- the block's histories regrouped into spatially
 * compact tubes whose x / {Delta, s} windows live in shared memory -- and smaller blocks the direct
 * kernel (one warp per history, gathers and reductions in L2); mode 1 = direct kernel only; mode 2 = plan
 * whenever it can be built.  The result is the same up to FP32 summation order (R18, R21). */
int pct_solve_config(pct_ctx* ctx, int mode, int64_t min_block);

/* Statistics of the solve plan cached in `paths` by the last pct_solve that used one (all zero if none). */
typedef struct {
    int64_t block_size, n_blocks, n_groups, n_direct, plan_bytes;
    /* what one sweep of the windowed kernel moves (bench.py's roofline): bytes of the slab-aligned code stream and of the
     * per-(slab, thread) visit counts (HBM, read once per pass), window slots staged from x / flushed to the
     * accumulator per sweep (L2 gathers / reductions that remain after the shared-memory aggregation), and the
     * histories and visits that take the windowed kernel */
    int64_t stream_bytes, cnt_bytes, staged_slots, windowed_histories, windowed_visits;
} pct_plan_stats;
int pct_plan_info(const pct_paths* paths, pct_plan_stats* out /* HOST */);

/* Per-kernel timing for the roofline report.  pct_profile_enable(ctx, 1) makes the launchers bracket every launch
 * of the hot kernels with CUDA events on the launching stream; pct_profile_read synchronises the device,
 * ADDS the elapsed times since the last read to out (HOST) and clears the event list.  kind: 0 = MLP + walk (K1),
 * 1 = windowed block projection (K2w), 2 = voxel update (K3), 3 = direct block projection (K2d),
 * 4 = solve-plan construction (sort, grouping, verification), 5 = preprocessing (pct_fbp, pct_hull_carve). */
#define PCT_PROFILE_KINDS 6
typedef struct {
    double ms[PCT_PROFILE_KINDS];
    int64_t launches[PCT_PROFILE_KINDS];
} pct_profile;
int pct_profile_enable(pct_ctx* ctx, int on);
int pct_profile_read(pct_ctx* ctx, pct_profile* out);

/* Roofline denominators MEASURED_PEAKS.json lacks, measured on ctx's device with register /
 * L2 / shared-memory resident microbenchmarks (best of three launches, CUDA events; ~0.3 s in total):
 * plain FP64 FMA/s (K1), random 4-byte L2 gathers/s over a 64 MiB array, red.global.add.f32/s and .v2.f32/s
 * (random and warp-contiguous addresses), shared-memory 32-bit atomic adds/s and loads/s (random slots, and
 * conflict-free).
 * out: HOST.  Blocking; uses the legacy default stream. */
typedef struct {
    double fp64_fma_per_s, l2_gather_per_s, l2_red_f32_per_s, l2_red_v2_per_s, l2_red_v2_coalesced_per_s,
        smem_atomic_per_s, smem_load_per_s;          /* random slots: the bank conflicts of an arbitrary address stream */
    double smem_atomic_cf_per_s, smem_load_cf_per_s; /* conflict-free (lane l -> bank l): the pipe's own ceiling        */
    int32_t num_sms;
} pct_peaks;
int pct_measure_peaks(pct_ctx* ctx, pct_peaks* out);

#ifdef __cplusplus
}
#endif
#endif
