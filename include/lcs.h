/* lcs.h -- C-ABI of liblcs.so: the B200 (sm_100a) hot path of the LCS pipeline of arXiv 2209.13775.
 *
 *   velocity snapshots on a mesh --lcs_field_create/lcs_field_set_snapshot--> resident field
 *   seeds --lcs_advect (RK4, Eq. 1.2)--> flow map F_{t0}^{tf} + exit flags
 *   flow map --lcs_cg_ftle (central differences, Eq. 1.1)--> Cauchy-Green tensor C, FTLE
 *   positions --lcs_locate--> containing mesh cell
 *
 * Conventions
 *  - Plain C, no exceptions or aborts cross the boundary; every call returns an lcs_status and
 *    lcs_last_error() gives a thread-local message.  A tracer leaving the domain is DATA (flags).
 *  - "device" pointers are CUDA device pointers of the current device, allocated and owned by the
 *    caller (the Python binding uses torch tensors); "host" pointers are ordinary memory.  The library
 *    owns only what lives behind lcs_field (mesh, snapshots, tracer scratch).
 *  - The hot calls (lcs_locate, lcs_advect, lcs_cg_ftle) are asynchronous on `cuda_stream` (a
 *    cudaStream_t passed as void*, NULL = default stream); the caller synchronises.  They never allocate or
 *    free device memory and never synchronise the device: everything lcs_advect needs is allocated by
 *    lcs_field_reserve (a set-up call), and lcs_advect returns LCS_ERR_OOM if the reservation is too small.
 *  - Every step of the path runs in CUDA kernels; there is no CPU fallback.
 *  - A field owns one set of tracer scratch buffers and one snapshot window: run one hot call at a time per field
 *    (calls on the same stream serialise by themselves); different fields are independent.
 * Citations are PAPER.md lines (the paper text) and DESIGN.md readings where the paper is silent.
 */
#ifndef LCS_H
#define LCS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lcs_field lcs_field;           /* opaque; owns device copies of mesh + snapshots */

typedef enum {
    LCS_OK = 0,
    LCS_ERR_INVALID_ARG = 1,
    LCS_ERR_TIME_RANGE = 2,                   /* [t0,tf] not inside the snapshot times            */
    LCS_ERR_MESH = 3,                         /* bad connectivity / index out of range            */
    LCS_ERR_OOM = 4,
    LCS_ERR_CUDA = 5,
    LCS_ERR_NOT_READY = 6                     /* a snapshot needed by the call was never set      */
} lcs_status;

typedef enum { LCS_F32 = 0, LCS_F64 = 1 } lcs_dtype;
typedef enum { LCS_MESH_CARTESIAN = 0, LCS_MESH_SIMPLEX = 1 } lcs_mesh_kind;

/* Description of gridded, time-sampled velocity data u(x,t): a Cartesian grid or a
 * simplicial mesh (triangles / tetrahedra) plus the snapshot times.               */
typedef struct {
    int32_t dim;                              /* 2 or 3                                           */
    int32_t kind;                             /* lcs_mesh_kind                                    */
    /* Cartesian: n[a] nodes on axis a, node i at origin[a] + i*spacing[a]; periodic[a] != 0 => n[a]
     * cells on that axis and node n[a] == node 0, else n[a]-1 cells.  Node index = i0 + n0*(i1 + n1*i2). */
    int32_t n[3];
    int32_t periodic[3];
    double origin[3];
    double spacing[3];
    /* Simplex: HOST pointers, copied during create.  vertices [n_vertices][dim] fp64; cells
     * [n_cells][dim+1] int32 of any orientation.  The library builds face adjacency and a uniform bin
     * grid on the device.                                                                          */
    int64_t n_vertices;
    int64_t n_cells;
    const double *vertices;
    const int32_t *cells;
    /* Time: strictly increasing and uniformly spaced, n_snapshots >= 2.  HOST pointer, copied.      */
    int32_t n_snapshots;
    int32_t vel_dtype;                        /* lcs_dtype: storage type of the velocity data     */
    const double *times;
    int32_t compute_dtype;                    /* lcs_dtype: type of seeds / flow map and of the
                                                 arithmetic inside lcs_advect                      */
    int32_t max_resident_snapshots;           /* 0 = keep every snapshot on the device; k >= 3 = ring of
                                                 k device slots fed from host memory on a side stream
                                                 (the temporal window of PAPER.md:57, 61, 85)      */
} lcs_field_desc;

/* Creates the field: uploads the mesh, orients cells, builds adjacency + bins (simplex).  Snapshots are
 * supplied afterwards.  *out is NULL on error.                                                     */
lcs_status lcs_field_create(const lcs_field_desc *desc, lcs_field **out);

/* Velocity of snapshot s (0-based), layout [node][dim] of vel_dtype, node order = mesh vertex order
 * (Cartesian: i0 fastest).  `vel` is a host pointer (pinned memory makes the copy asynchronous) or, with
 * is_device_ptr != 0, a device pointer.  The data is copied / re-laid-out on the library's side stream;
 * with max_resident_snapshots == 0 the caller may free `vel` after lcs_field_sync.  In ring mode the
 * HOST pointer is retained and must stay valid until lcs_field_destroy (snapshots are re-streamed
 * from it whenever the window moves; "loaded into GPU memory only when a new file is needed"). */
lcs_status lcs_field_set_snapshot(lcs_field *f, int32_t s, const void *vel, int32_t is_device_ptr);
lcs_status lcs_field_sync(lcs_field *f);
void lcs_field_destroy(lcs_field *f);

/* Set-up call: allocates everything lcs_advect / lcs_advect_early_cg need for up to n_seeds tracers and n_steps RK4
 * steps per call under the CURRENT options: tracer records and sort scratch, stage-time tables, the pair-record cache,
 * the blended stage-time fields of one chunk (3D fp32 Cartesian grids) and the resident field sets (option
 * "field_sets").  The paper loads velocity data into GPU memory "only every time a new velocity data file is needed"
 * (PAPER.md:85); nothing else may stall the stream, so the hot calls themselves never allocate.  Grow-only and
 * idempotent: a call that asks for no more than what is reserved returns at once; growing synchronises the device, frees
 * and re-allocates.  Options that change the footprint ("field_sets", "preblend_steps", "integrator", "bundle", "tma")
 * must be set BEFORE the reservation they are meant for; lcs_advect returns LCS_ERR_OOM ("call lcs_field_reserve") when
 * the reservation does not cover a call.  Errors: LCS_ERR_INVALID_ARG (n_seeds < 1, n_steps < 1, n_seeds >= 2^31,
 * n_steps >= 2^24), LCS_ERR_OOM.                                                                                  */
lcs_status lcs_field_reserve(lcs_field *f, int64_t n_seeds, int64_t n_steps);

/* Integer options.  Keys: "integrator" 0 = auto, 1 = fused (one persistent per-seed loop per snapshot
 * window), 2 = split (the paper's design: tracers advance synchronously, one short kernel per RK4 stage on Cartesian grids, one per
 * cell search and one per interpolation -- 8 launches per step -- on simplicial meshes: PAPER.md:85-87), 3 = 4-step
 * Adams-Bashforth with three RK4 start-up steps ("Adams-Bashforth (multi-step)"; one velocity evaluation per step);
 * "bundle" -1 = auto, 0 = off, 1 = on: re-bundle tracers by cell (Morton order of the cell index) so that a
 * warp gathers from neighbouring cells; results are returned in the caller's order;
 * "bundle_steps" k = re-bundle every k RK4 steps (0 = once per snapshot window; unstructured meshes: every 160 steps);
 * "bundle_order" / "simplex_order" 0 = Morton, 1 = row-major (x fastest) sort key over cells / bins; "bundle_order" -1 (default) = Morton for the
 * pre-blended integrator, row-major otherwise; "simplex_order" defaults to 1 ("bundle_order" 2 = pairs of
 * x-neighbouring cells split by sub-cell octant, 3 = bricks of 4 x 2 x 2 cells; both 3D Cartesian only);
 * "field_sets" m = keep the blended fields of the last m chunks resident (about 7 GB each for a 128^3 grid and 50-step chunks)
 * and reuse them when a later lcs_advect needs the same snapshot pair and stage times (FTLE time series: volumes released one
 * snapshot interval apart share most windows); "field_sets_clear" = forget them;
 * "preblend" -1/0/1 and "preblend_steps" k: 3D fp32 Cartesian grids gather from per-stage-time blended fields, k steps per launch;
 * "tma" 0/1/2 (default 0): 3D fp32 grids that are periodic with power-of-two node counts on every axis: the pre-blended integrator
 * stages the records of each block's bounding box through shared memory with TMA bulk copies (cp.async.bulk + mbarrier), tracers
 * bundled in 4 x 2 x 2-cell bricks (2: in the order of "bundle_order"); bit-identical results; measured SLOWER than the global-memory
 * gather on B200 (profiles/r2_cfg3_tma.md), hence off by default; "tma_cap" = records per shared-memory tile (default 704);
 * "ld256" 0/1 = gather each 32-byte node record with one 256-bit load; "block" = threads per block;
 * "time_windows" 0/1 = record CUDA events around the integrator launches (read with lcs_field_get_info). */
lcs_status lcs_field_set_option(lcs_field *f, const char *key, int64_t value);
/* Counters and sizes.  Keys: "n_nodes", "n_cells", "n_bins", "n_boundary_faces" (mesh); "ring", "windows" (snapshot windows visited),
 * "h2d_bytes" (snapshot bytes uploaded so far), "scratch_bytes" (reserved tracer scratch); "locate_fallbacks", "locate_random_walks",
 * "locate_hops", "locate_max_hops" (canonical walks of lcs_locate and of the seeds; the first two stay 0 on the seeded inputs),
 * "walk_fallbacks" (in-advect walks that gave up and were re-located with the canonical predicate), "walk_cap_hits" (tracers
 * interpolated in a cell that does not hold them: 0 by construction); "field_set_hits", "field_set_misses"; "series_layers" (batched
 * layers of the last lcs_advect_series, 0 = integrated volume by volume); "window_launches", "window_time_ns" (with option
 * "time_windows": integrator launches bracketed by CUDA events and their summed duration; reading the latter synchronises).
 * Errors: LCS_ERR_INVALID_ARG for an unknown key.                                                                            */
lcs_status lcs_field_get_info(const lcs_field *f, const char *key, int64_t *value);

/* Cell containing each position ("computes which cell ... each seed point is located in";
 * PAPER.md:87 cell search).  pos: device [n][dim] fp64.  cell: device [n] int32, -1 = outside.
 * Cartesian: arithmetic indexing, cell id = i0 + nc0*(i1 + nc1*i2), upper boundary closed.
 * Simplex: bin grid -> start cell -> walk across faces with the canonical fp64 face predicate (vertices
 * of a face sorted by id, every product and sum rounded separately, ties broken as if the point were
 * p + (eps, eps^2, eps^3)); the result is the unique owner, bit-exact against the oracle.
 * bary (optional, may be NULL): device [n][dim] Cartesian weights or [n][dim+1] barycentric weights.
 * Simplicial meshes are taken to triangulate a CONVEX region (Delaunay triangulations do; reading #11): a walk that
 * reaches a hull face with the point strictly beyond it reports "outside" (-1; in lcs_advect: exit flag 1), so a point that is
 * inside the mesh but separated from the walk's start by a concavity or a hole may be reported as outside.              */
lcs_status lcs_locate(lcs_field *f, int64_t n, const double *pos, int32_t *cell, double *bary,
                      void *cuda_stream);

/* Flow map by classical RK4 of dx/dt = u(x,t) (Eq. 1.2) with bi/trilinear or
 * barycentric interpolation in space and linear interpolation in time between the two bracketing
 * snapshots.  N = round((tf-t0)/h) steps; h < 0 integrates backward in time.
 * seeds, flowmap: device [n][dim] of compute_dtype; flowmap may alias seeds.
 * exit_flag (device [n] u8, may be NULL): 0 = inside the domain up to tf; 1 = left during integration
 *   (any of the four RK4 evaluation points outside; flowmap = position at the start of that step;
 *   PAPER.md:65); 2 = seed outside at t0 (flowmap = seed).
 * exit_step (device [n] i32, may be NULL): completed steps (N for flag 0, 0 for flag 2).
 * Errors: LCS_ERR_INVALID_ARG if h == 0, sign(h) != sign(tf-t0) or |N*h-(tf-t0)| > 1e-9*|tf-t0|;
 * LCS_ERR_TIME_RANGE if [t0,tf] leaves [times[0], times[ns-1]] by more than 1e-9 snapshot intervals.   */
lcs_status lcs_advect(lcs_field *f, int64_t n, const void *seeds, double t0, double tf, double h,
                      void *flowmap, uint8_t *exit_flag, int32_t *exit_step, void *cuda_stream);

/* FTLE time series: the same n seeds released at n_vol times t_start[k] (HOST array) and each integrated over the signed interval T
 * with step h, i.e. n_vol calls of lcs_advect(seeds, t_start[k], t_start[k] + T, h) (LCS are followed through time as a
 * sequence of FTLE fields; the cached window of velocity frames serves every tracer that is inside it).
 * flowmaps: device [n_vol][n][dim] of compute_dtype; exit_flags (may be NULL): device [n_vol][n] u8; exit_steps (may be NULL):
 * device [n_vol][n] i32; per volume exactly what lcs_advect returns (bit for bit: a tracer's arithmetic does not depend on who
 * shares its launch).  On 3D fp32 Cartesian grids whose volumes are the same integration shifted by whole snapshot intervals the
 * volumes that are inside a snapshot window at the same time are advanced TOGETHER -- one blend of the window's stage-time fields
 * and one integrator launch over the tracers of all of them, bundled by cell; otherwise the volumes are integrated one after the
 * other.  lcs_advect_series_reserve is the set-up call (the series needs room for the tracers of all overlapping volumes plus one;
 * option "field_sets" must be 0).  n_vol * n < 2^31.  Errors as lcs_advect; LCS_ERR_OOM without a covering reservation.        */
lcs_status lcs_advect_series_reserve(lcs_field *f, int64_t n, int32_t n_vol, const double *t_start, double T, double h);
lcs_status lcs_advect_series(lcs_field *f, int64_t n, const void *seeds, int32_t n_vol, const double *t_start, double T, double h,
                             void *flowmaps, uint8_t *exit_flags, int32_t *exit_steps, void *cuda_stream);

/* Central-difference flow-map gradient G_ab = dF_a/dx_b on the structured seed grid,
 * Cauchy-Green tensor C = G^T G (Eq. 1.1), its largest eigenvalue (closed form) and
 * FTLE = ln(lambda_max) / (2|T|), fused in one kernel.
 * Seed index = i0 + ng0*(i1 + ng1*i2); seed_spacing per axis; seed_periodic[a] != 0 => differences wrap
 * on that axis, adding +-period[a] to component a of the wrapped neighbour.
 * flowmap: device [n][dim] of `dtype`; exit_flag: device [n] u8 or NULL (all valid).
 * A neighbour is valid if it is inside the grid (or reached by wrap) and its flag is 0.  Both valid:
 * central difference; one valid and the seed valid: one-sided, status bit 1; seed invalid or no valid
 * neighbour on some axis: C, FTLE = NaN, status bit 0.
 * cg: device [n][3] (C11,C12,C22) or [n][6] (C11,C12,C13,C22,C23,C33) of `dtype`, may be NULL.
 * ftle: device [n] of `dtype`.  status: device [n] u8, may be NULL.  Arithmetic is fp64 throughout. */
lcs_status lcs_cg_ftle(int32_t dim, int32_t dtype, const int32_t ng[3], const double seed_spacing[3],
                       const int32_t seed_periodic[3], const double period[3],
                       const void *flowmap, const uint8_t *exit_flag, double T,
                       void *cg, void *ftle, uint8_t *status, void *cuda_stream);

/* Flow map WITH early evaluation of the Cauchy-Green tensor (when a tracer leaves the domain "the
 * computation of the CG tensor is performed" for the stencils it belongs to instead of discarding them; PAPER.md:85, 153:
 * all tracers advance together, so C "can be evaluated at any time step").  Same integration as lcs_advect on the
 * structured seed grid ng (n = ng0*ng1*ng2 seeds, layout as in lcs_cg_ftle).  Evaluation points are the step counts
 * m = every, 2*every, ... and N.  At m a seed is (re-)evaluated iff it has completed m steps and none of its 2*dim grid
 * neighbours has left; neighbours that never started (flag 2) or lie outside the grid are invalid neighbours as in
 * lcs_cg_ftle (one-sided differences).  The evaluation is that of lcs_cg_ftle with T_eff = m*h.  A seed keeps the
 * result of its last evaluation: t_eff[n] (compute_dtype) is m*h of it, 0 if it was never evaluated (then C, FTLE = NaN,
 * status bit 0).  flowmap / exit_flag / exit_step: as lcs_advect (flowmap and exit_flag are required and must not alias
 * seeds: they are rewritten at every evaluation point).  cg and status may be NULL.  every >= 1.                  */
lcs_status lcs_advect_early_cg(lcs_field *f, const int32_t ng[3], const double seed_spacing[3],
                               const int32_t seed_periodic[3], const double period[3], const void *seeds,
                               double t0, double tf, double h, int32_t every, void *flowmap, uint8_t *exit_flag,
                               int32_t *exit_step, void *cg, void *ftle, void *t_eff, uint8_t *status,
                               void *cuda_stream);

/* Cauchy-Green tensor and FTLE from AUXILIARY points instead of neighbouring seeds ("a structured grid
 * of auxiliary points can be placed around each seed point"; the Cauchy-Green filter uses them "for the
 * computation of the flow map gradient").  The caller advects, with lcs_advect, 2*dim auxiliary tracers per seed released
 * at x0 + aux_delta[b] e_b (entry 2b) and x0 - aux_delta[b] e_b (entry 2b+1).
 * flowmap_aux: device [n][2*dim][dim] of `dtype`; exit_flag_aux: device [n][2*dim] u8 or NULL.
 * G_ab = (F_a(+b) - F_a(-b)) / (2 aux_delta[b]), always central; a seed with any flagged auxiliary tracer gets
 * C, FTLE = NaN and status 1.  cg / ftle / status as in lcs_cg_ftle.  Errors: aux_delta[b] <= 0, T == 0.          */
lcs_status lcs_cg_ftle_aux(int32_t dim, int32_t dtype, int64_t n, const double aux_delta[3], const void *flowmap_aux,
                           const uint8_t *exit_flag_aux, double T, void *cg, void *ftle, uint8_t *status,
                           void *cuda_stream);

/* All eigenvalues and eigenvectors of the Cauchy-Green tensor (the Cauchy-Green filter attaches
 * "eigenvalues and eigenvectors"; hyperbolic-LCS criteria use the eigenvector fields).  Cyclic Jacobi
 * in fp64 per seed (reading #27).  cg: device [n][3] or [n][6] of `dtype` as written by lcs_cg_ftle.
 * evals: device [n][dim], ascending.  evecs: device [n][dim][dim], row i = unit eigenvector of evals[i], its component
 * of largest magnitude positive.  A seed whose C holds a non-finite value gets NaN in both outputs.                */
lcs_status lcs_cg_eigen(int32_t dim, int32_t dtype, int64_t n, const void *cg, void *evals, void *evecs,
                        void *cuda_stream);

/* Gaussian smoothing of a scalar field (the FTLE) on the structured seed grid, the first step of the LCS filter
 * ("Gaussian smoothing of FTLE" before ridge extraction; reading #30).  One normalised 1D convolution
 * per axis, axis 0 first: out(i) = sum_k w_k f(i+k) / sum_k w_k over |k| <= ceil(3 sigma) with f(i+k) finite and inside the grid
 * (wrapped on a periodic axis), w_k = exp(-k^2 / (2 sigma^2)), sigma in seed-grid cells, 0 < sigma <= 21.33.  A NaN centre
 * stays NaN; NaN neighbours are skipped.  field, out, work: three distinct device buffers of [n] `dtype` (work is scratch). */
lcs_status lcs_smooth_gaussian(int32_t dim, int32_t dtype, const int32_t ng[3], const int32_t seed_periodic[3],
                               double sigma, const void *field, void *out, void *work, void *cuda_stream);

/* lcs_smooth_gaussian for callers that cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same passes, same results, but the intermediate field lives in a file-scope device array of the library
 * instead of a caller-supplied work buffer, and the call allocates and frees nothing (no cudaMalloc / cudaFree, no allocating
 * library routine; the array's device address is looked up once per device).  Limit: ng0*ng1*ng2 * sizeof(dtype) <= 16 MiB, i.e.
 * 4 194 304 fp32 or 2 097 152 fp64 seeds; larger grids return LCS_ERR_INVALID_ARG (use lcs_smooth_gaussian).  Every GPU that loads
 * the library holds the 16 MiB until the process exits.  All calls on a device share the array, which keeps the last call's contents
 * (nothing in it has to start at zero: each pass reads only what the pass before wrote): calls that overlap on the GPU -- different
 * streams, or different host threads -- race on it; calls on one stream serialise by themselves.
 * field, out: two distinct device buffers of [n] `dtype`.  Other arguments and errors as lcs_smooth_gaussian.                  */
lcs_status lcs_smooth_gaussian_static(int32_t dim, int32_t dtype, const int32_t ng[3], const int32_t seed_periodic[3],
                                      double sigma, const void *field, void *out, void *cuda_stream);

/* Ridge indicator of a scalar field (the smoothed FTLE) on the structured seed grid, the second step of the LCS filter
 * ("C-ridge extraction"; the paper gives no definition: DESIGN.md reading #32, second-derivative ridge).
 * Per seed: gradient g and Hessian H by central differences on the 3^dim stencil (wrapped on periodic axes), kappa = smallest
 * eigenvalue of H with unit eigenvector n (component of largest magnitude positive), d = g . n,
 * mask = (kappa < -kappa_min) && (field >= s_min) && (|d| <= |kappa| * min(seed_spacing) / 2): the ridge passes within half
 * a cell of the seed.  A seed whose stencil leaves a non-periodic grid or holds a non-finite value gets kappa = d = NaN,
 * mask = 0.  field, kappa, dgn: device [n] of `dtype`; mask: device [n] u8.  fp64 arithmetic.  kappa_min >= 0.          */
lcs_status lcs_ridge(int32_t dim, int32_t dtype, const int32_t ng[3], const double seed_spacing[3],
                     const int32_t seed_periodic[3], double kappa_min, double s_min, const void *field,
                     void *kappa, void *dgn, uint8_t *mask, void *cuda_stream);

/* End-to-end convenience with HOST buffers: copies the seeds to the device, runs lcs_advect and
 * lcs_cg_ftle and copies the flow map, flags, exit steps, Cauchy-Green tensor (each optional, NULL = not
 * wanted) and the FTLE back; synchronous (it reserves what it needs: lcs_field_reserve + its own staging).
 * seeds_host/flowmap_host: [n][dim] of the field's compute_dtype; cg_host: [n][3 or 6]; ftle_host: [n] of
 * compute_dtype; exit_flag_host [n] u8; exit_step_host [n] i32.
 * Pinned host memory makes the copies asynchronous with respect to each other.                      */
lcs_status lcs_ftle_host(lcs_field *f, const int32_t ng[3], const double seed_spacing[3],
                         const int32_t seed_periodic[3], const double period[3],
                         const void *seeds_host, double t0, double tf, double h,
                         void *flowmap_host, uint8_t *exit_flag_host, int32_t *exit_step_host,
                         void *cg_host, void *ftle_host);

/* The time-series counterpart of lcs_ftle_host: seeds up, lcs_advect_series, lcs_cg_ftle per volume, results down; synchronous.
 * t_start: HOST [n_vol].  Outputs are [n_vol][n]... arrays in HOST memory: ftle_host [n_vol][n] (required); flowmaps_host
 * [n_vol][n][dim], exit_flags_host [n_vol][n], exit_steps_host [n_vol][n], cg_host [n_vol][n][3 or 6] (each optional).   */
lcs_status lcs_ftle_series_host(lcs_field *f, const int32_t ng[3], const double seed_spacing[3], const int32_t seed_periodic[3],
                                const double period[3], const void *seeds_host, int32_t n_vol, const double *t_start, double T, double h,
                                void *flowmaps_host, uint8_t *exit_flags_host, int32_t *exit_steps_host, void *cg_host, void *ftle_host);

/* Measured peaks of the device the roofline fractions are quoted against ("Peaks to measure on the box
 * before quoting any %"; the paper's claim under test is "limited by memory bandwidth").  Runs a
 * micro-kernel (warm-up + best of 3, CUDA events), synchronous, allocates and frees its own buffers (up to 2 GB).
 * value: TFLOP/s for the FMA kinds, microseconds for LCS_PEAK_LAUNCH_US, GB/s otherwise (bytes delivered to registers for
 * the gather kinds: 32 bytes per lane and load).                                                                   */
typedef enum {
    LCS_PEAK_FP32_FMA = 0,            /* dependent-free FFMA chains, all SMs                                        */
    LCS_PEAK_FP64_FMA = 1,
    LCS_PEAK_LAUNCH_US = 2,           /* back-to-back empty kernel launches, microseconds per launch                */
    LCS_PEAK_HBM_COPY = 3,            /* 1 GiB streaming copy, read + write bytes                                   */
    LCS_PEAK_L2_SEQ = 4,              /* sequential 128-bit reads of a 48 MB buffer, L1 bypassed                    */
    LCS_PEAK_L2_SECTOR = 5,           /* random 32-byte sectors of a 32 MB buffer (L2-resident), L1 bypassed        */
    LCS_PEAK_HBM_SECTOR = 6,          /* random 32-byte sectors of a 2 GB buffer                                    */
    LCS_PEAK_L1_GATHER_LINE = 7,      /* L1-resident 256-bit gathers, the 4 lanes of a group read one 128-byte line */
    LCS_PEAK_L1_GATHER_SAME = 8,      /* ... the 4 lanes of a group read the same 32-byte record                    */
    LCS_PEAK_L1_GATHER_SPREAD = 9,    /* ... every lane reads a line of its own                                     */
    LCS_PEAK_SMEM_CONTIGUOUS = 10,    /* shared memory, LDS.128, lane L reads chunk base + L (conflict-free)        */
    LCS_PEAK_SMEM_RECORDS = 11,       /* shared memory, lane L reads the 32-byte record base + L as 2 x LDS.128     */
    LCS_PEAK_SMEM_RECORDS_SWIZZLED = 12, /* ... with the 16-byte chunks laid out as TMA's 32-byte swizzle does      */
    LCS_PEAK_SMEM_RECORDS_SAME = 13,  /* ... swizzled, the 4 lanes of a group read the same record (broadcast)      */
    LCS_PEAK_L1_GATHER_WARP_SAME = 14,   /* L1-resident 256-bit gathers, the whole warp reads one record             */
    LCS_PEAK_L1_GATHER_WARP_LINE = 15,   /* ... the whole warp reads the four records of one 128-byte line           */
    LCS_PEAK_L1_GATHER_WARP_2LINES = 16  /* ... two lines, 16 lanes each                                             */
} lcs_peak_kind;
lcs_status lcs_measure_peak(int32_t kind, double *value);

/* Number of kernels this library has launched in this process (bench.py's gpu_launches).           */
int64_t lcs_kernel_launch_count(void);

const char *lcs_last_error(void);             /* thread-local, static storage                       */

#ifdef __cplusplus
}
#endif
#endif /* LCS_H */
