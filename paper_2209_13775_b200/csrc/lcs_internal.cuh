// lcs_internal.cuh -- private declarations of liblcs.so (sm_100a).  Not part of the C-ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include <string>
#include <vector>

#include "../../include/lcs.h"

// ---------------------------------------------------------------------------------------------
// error plumbing
void lcs_set_error(const char *fmt, ...);
extern std::atomic<int64_t> g_lcs_launches;

#define LCS_CUDA_OK(expr)                                                                       \
    do {                                                                                        \
        cudaError_t e__ = (expr);                                                               \
        if (e__ != cudaSuccess) {                                                               \
            lcs_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return (e__ == cudaErrorMemoryAllocation) ? LCS_ERR_OOM : LCS_ERR_CUDA;             \
        }                                                                                       \
    } while (0)

#define LCS_LAUNCH(kernel, grid, block, smem, stream, ...)                                      \
    do {                                                                                        \
        kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);                             \
        g_lcs_launches.fetch_add(1, std::memory_order_relaxed);                                 \
    } while (0)

static inline unsigned lcs_blocks(int64_t n, int block) { return (unsigned)((n + block - 1) / block); }

// ---------------------------------------------------------------------------------------------
// Velocity "pair record": for one mesh node, the velocity at the earlier snapshot of the current window
// (a) and the difference to the later one (d = b - a), padded to P = 2 (2D) or 4 (3D) components.
// u(node, tau) = a + tau*d is one FMA per component, and both time levels of a node share one 32-byte
// sector for the two hot layouts (3D fp32, 2D fp64).
template <int DIM> struct PadOf { static constexpr int P = (DIM == 2) ? 2 : 4; };

template <int DIM, typename TV> struct alignas(16) PairRec {
    TV a[PadOf<DIM>::P];
    TV d[PadOf<DIM>::P];
};

// ---------------------------------------------------------------------------------------------
struct CartGeom {
    int32_t n[3];          // nodes per axis
    int32_t np[3];         // padded record counts per axis: n + 1.  Rows are deliberately NOT rounded up to whole 128-byte lines:
                           // measured on config 3, a row stride of 132 instead of 129 records costs 17% (L1 set conflicts between
                           // the four rows a stage gathers from)
    int32_t periodic[3];
    int32_t pow2[3];       // n[a] is a power of two (mask wrap)
    double origin[3];
    double spacing[3];
    double inv[3];         // 1.0 / spacing, rounded once (oracle O2)
};

struct SimplexMesh {
    int64_t nv = 0, nc = 0;
    double *verts = nullptr;      // [nv][dim] fp64
    int32_t *cells = nullptr;     // [nc][dim+1]
    int32_t *neigh = nullptr;     // [nc][dim+1], -1 = hull face
    uint8_t *oppside = nullptr;   // [nc] bit j = canonical side of the vertex opposite face j
    void *cellrec = nullptr;      // [nc] per-cell affine map for the in-advect walk (compute dtype)
    int32_t *bins = nullptr;      // [nb0*nb1*nb2] start cell per bin
    int32_t nb[3] = {1, 1, 1};
    double bin_lo[3] = {0, 0, 0};
    double bin_inv[3] = {0, 0, 0};
    int64_t hop_cap = 64;
    unsigned long long *stats = nullptr;   // [0] brute-force fallbacks, [1] walk hops, [2] max hops of one walk (lcs_locate + seeds),
                                           // [3] random-walk fallbacks, [4] in-advect walks that ended in a cell not holding the point
                                           // (0 by construction), [5] in-advect walks re-located with the canonical predicate,
                                           // [8..11] as [0..3] for those re-locations
};

// tracer scratch owned by the field: one allocation made by lcs_field_reserve and carved by the advect code
struct TracerScratch {
    void *buf = nullptr;
    size_t bytes = 0;
    int64_t n_seeds = 0, n_steps = 0;     // what the last lcs_field_reserve asked for
};

// context of lcs_advect_early_cg (row f1): where and when the integrators evaluate C during the advection
struct EarlyCg {
    bool on = false;
    int64_t every = 0;            // evaluation points: step counts that are multiples of `every`, and N
    int32_t ng[3] = {1, 1, 1}, per[3] = {0, 0, 0};
    double dx[3] = {1, 1, 1}, period[3] = {0, 0, 0};
    double h = 0;
    void *flowmap = nullptr, *cg = nullptr, *ftle = nullptr, *t_eff = nullptr;
    uint8_t *flag = nullptr, *status = nullptr;
};

// A resident set of blended x-pair fields (one chunk of the pre-blended integrator): FTLE time series release one seed grid
// per snapshot interval, and consecutive volumes share nine tenths of their stage times; with 180 GB of HBM the sets of the
// last windows stay resident and are reused instead of blended again (option "field_sets" = how many to keep, 0 = off).
struct FieldSet {
    int pair = -1;                // snapshot pair the set was blended from
    std::vector<float> tau;       // stage-time weights of its fields, compared exactly
    void *buf = nullptr;
    size_t bytes = 0;
    int64_t age = 0;
};

struct lcs_field {
    lcs_field() { for (int k = 0; k < kMaxPairCache; ++k) pair_snap[k] = -1; }
    int dim = 0, kind = 0;
    int vel_dtype = 0, compute_dtype = 0;
    int P = 2;                    // padded components
    int64_t nnodes = 0;
    int64_t nrec = 0;             // pair records per window buffer (Cartesian: np[0] * np[1] * np[2])
    CartGeom cart{};
    SimplexMesh mesh{};
    std::vector<double> times;
    double dt_snap = 0;
    int ns = 0;
    // snapshot storage: raw slots hold [node][dim] of vel dtype exactly as supplied
    int nslots = 0;
    bool ring = false;
    std::vector<void *> slot;            // device buffers
    std::vector<int> slot_snap;          // snapshot held (or being loaded) in slot, -1 = empty
    std::vector<cudaEvent_t> slot_ready; // recorded on the side stream after the upload
    std::vector<cudaEvent_t> slot_free;  // recorded on the compute stream after the last reader
    std::vector<char> slot_free_valid;
    std::vector<int> snap_slot;          // slot of snapshot s, -1 = not resident
    std::vector<char> snap_set;
    std::vector<const void *> host_src;  // ring mode: retained host pointers
    // pair-record cache (built on the compute stream from two raw slots)
    // 4 entries (a window and its neighbours), or one per snapshot pair when the whole series of pair records fits 256 MB
    // (small fields: configs 1 and 2 then build every pair once instead of once per pass)
    static constexpr int kMaxPairCache = 64;
    int n_pair_cache = 4;
    void *pair_buf[kMaxPairCache] = {};
    int pair_snap[kMaxPairCache];
    int64_t pair_age[kMaxPairCache] = {};
    int64_t pair_clock = 0;
    cudaStream_t side = nullptr;
    TracerScratch scratch;
    // host-API scratch
    void *h_seeds = nullptr, *h_flow = nullptr, *h_ftle = nullptr, *h_cg = nullptr;
    void *hs_flow = nullptr, *hs_ftle = nullptr, *hs_cg = nullptr;      // staging of lcs_ftle_series_host ([n_vol][n] arrays)
    uint8_t *hs_flag = nullptr;
    int32_t *hs_step = nullptr;
    int64_t hs_cap = 0;
    uint8_t *h_flag = nullptr;
    int32_t *h_step = nullptr;
    int64_t h_cap = 0;
    EarlyCg early;
    std::vector<FieldSet> field_sets;
    int64_t field_set_clock = 0, info_field_set_hits = 0, info_field_set_misses = 0;
    // options
    int64_t opt_integrator = 0;   // 0 auto, 1 fused, 2 split
    int64_t opt_bundle = -1;      // re-bundle tracers by cell: -1 auto (large seed sets), 0 off, 1 on
    int64_t opt_bundle_order = -1; // Cartesian sort key: -1 = auto (Morton for the pre-blended integrator, whose gathers bypass L1 allocation and live on L2
                                   // locality; row-major otherwise), 0 = Morton code of the cell, 1 = row-major cell index (x fastest), 2 / 3: see lcs.h
    int64_t opt_simplex_order = 1; // simplex sort key over the bin grid: 0 = Morton, 1 = row-major
    int64_t opt_bundle_steps = 0; // RK4 steps between re-bundlings (0 = once per snapshot window)
    int64_t opt_preblend = -1;    // 3D fp32 Cartesian: gather from per-stage-time blended fields (-1 auto, 0 off, 1 on)
    int64_t opt_preblend_steps = 50; // RK4 steps per launch of the pre-blended integrator (2k+1 blended fields resident)
    int64_t opt_field_sets = 0;   // number of resident blended-field sets (0 = blend every chunk into scratch)
    int64_t opt_tma = 0;          // 3D fp32 periodic power-of-two grids: stage the blended fields through shared memory with TMA bulk copies
    int64_t opt_tma_cap = 704;    // records per shared-memory tile of the staged variant (2 tiles per block)
    int64_t opt_ld256 = 1;        // gather pair records with one 256-bit load instead of two 128-bit loads
    int64_t opt_block = 0;        // threads per block override (0 = default)
    int64_t opt_time_windows = 0; // record CUDA events around every window (hot) kernel launch
    // info
    int64_t info_windows = 0;
    int64_t info_series_layers = 0;      // batched layers of the last lcs_advect_series (0: integrated volume by volume)
    int64_t info_h2d_bytes = 0;
    std::vector<cudaEvent_t> win_ev;     // start/stop pairs recorded on the launching stream
    size_t win_ev_used = 0;
};

// CUDA-event bracket around the dominant kernel's launches (bench.py's roofline.achieved)
struct WindowTimer {
    lcs_field *f; cudaStream_t st; bool on;
    WindowTimer(lcs_field *f_, cudaStream_t st_) : f(f_), st(st_), on(f_->opt_time_windows != 0) {
        if (!on) return;
        while (f->win_ev.size() < f->win_ev_used + 2) { cudaEvent_t e; cudaEventCreate(&e); f->win_ev.push_back(e); }
        cudaEventRecord(f->win_ev[f->win_ev_used], st);
    }
    ~WindowTimer() { if (on) { cudaEventRecord(f->win_ev[f->win_ev_used + 1], st); f->win_ev_used += 2; } }
};

static inline size_t lcs_esize(int dtype) { return dtype == LCS_F64 ? 8 : 4; }

// field.cu
lcs_status lcs_field_require_pair(lcs_field *f, int s, cudaStream_t stream, const void **pair);
lcs_status lcs_field_prefetch(lcs_field *f, int s, int keep0, int keep1);
lcs_status lcs_field_acquire_raw(lcs_field *f, int s, cudaStream_t stream, const void **a, const void **b);
lcs_status lcs_field_release_raw(lcs_field *f, int s, cudaStream_t stream);
// lcs_advect never allocates: it checks that lcs_field_reserve made the scratch large enough (LCS_ERR_OOM otherwise)
lcs_status lcs_scratch_check(lcs_field *f, size_t bytes);

// cg_ftle.cu: evaluate C for the stencils that are still complete after m steps (flow map + flags already scattered)
lcs_status lcs_early_cg_eval(lcs_field *f, int64_t m, cudaStream_t st);
// number of steps of a launch unit that starts at step `first` and would run `count` steps: cut at the next evaluation point
static inline int lcs_early_cut(const lcs_field *f, int64_t first, int count)
{
    if (!f->early.on) return count;
    int64_t next = (first / f->early.every + 1) * f->early.every;
    return (int)(next - first < count ? next - first : count);
}
static inline bool lcs_early_due(const lcs_field *f, int64_t end, int64_t N) { return f->early.on && (end % f->early.every == 0 || end == N); }

// simplex.cu
lcs_status lcs_simplex_build(lcs_field *f, const double *verts_host, const int32_t *cells_host);
void lcs_simplex_free(lcs_field *f);
lcs_status lcs_simplex_locate(lcs_field *f, int64_t n, const double *pos, int32_t *cell, double *bary, cudaStream_t st);
lcs_status lcs_simplex_advect(lcs_field *f, int64_t n, const void *seeds, double t0, double h, int64_t N,
                              void *flowmap, uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st);

// advect_cart.cu
lcs_status lcs_cart_locate(lcs_field *f, int64_t n, const double *pos, int32_t *cell, double *w, cudaStream_t st);
lcs_status lcs_cart_advect_series(lcs_field *f, int64_t n, const void *seeds, int n_vol, const double *t_start, double h, int64_t N,
                                  void *flowmaps, uint8_t *exit_flags, int32_t *exit_steps, cudaStream_t st, int64_t *cap_records_out);
lcs_status lcs_cart_advect(lcs_field *f, int64_t n, const void *seeds, double t0, double h, int64_t N,
                           void *flowmap, uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Window plan shared by the Cartesian and simplex integrators: consecutive RK4 steps whose three stage
// times (ta, tb, tc) use the same snapshot pair are run by one launch.
struct StepWindow {
    int64_t first = 0;      // first step index
    int32_t count = 0;      // steps in the window
    int32_t s[3] = {0, 0, 0};   // snapshot pair index used by the stage times ta, tb, tc
};
lcs_status lcs_plan_windows(const lcs_field *f, double t0, double h, int64_t N, std::vector<StepWindow> &windows);
// time weight of stage k (0: ta, 1: tb, 2: tc) of step n in snapshot pair s: (t - times[s]) / (times[s+1] - times[s]) with
// t = t0 + (n + k/2) h by multiplication (fp64, exactly as the oracle computes it; the device tables are filled by
// lcs_fill_stage_tau with the same operations, rounded separately)
static inline double lcs_stage_tau(const lcs_field *f, double t0, double h, int64_t n, int k, int s)
{
    const double t = t0 + ((double)n + 0.5 * (double)k) * h;
    return (t - f->times[s]) / (f->times[s + 1] - f->times[s]);
}
// device tables, no host copy: tau[3 i + k] (TC = float or double) for the `count` steps from `first` of window w, and
// (is_blend) ftau[0 .. 2 count] = (float) tau of ta_0, tb_0, ta_1, tb_1, ..., tc_last for a chunk of the pre-blended integrator
lcs_status lcs_fill_stage_tau(const lcs_field *f, double t0, double h, int64_t first, int count, const int32_t s[3], void *tau,
                              float *ftau, cudaStream_t st);
// bytes lcs_advect carves out of the scratch for n seeds and N steps under the current options (the two integrators and
// lcs_field_reserve use the same function, so a reservation always covers the call it was made for)
size_t lcs_cart_scratch_bytes(const lcs_field *f, int64_t n, int64_t N);
lcs_status lcs_cart_tma_configure(lcs_field *f);   // opts the staged kernel into the shared memory its tile capacity needs
size_t lcs_simplex_scratch_bytes(const lcs_field *f, int64_t n, int64_t N);
size_t lcs_cart_field_set_bytes(const lcs_field *f, int64_t N);     // one resident set of blended fields (0: not applicable)
