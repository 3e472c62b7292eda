// field.cu -- lcs_field life cycle, the resident snapshot window (row a0), window planning and the
// C-ABI entry points that dispatch to the Cartesian / simplex kernels.
//
// Snapshot window (PAPER.md:57 Cache filter, "a window of velocity data frames (nominally two
// ...) are loaded on the GPU's memory", "velocity data is loaded into GPU memory only every
// time a new velocity data file is needed"): raw snapshots live in device slots (all of them, or a ring of
// k fed from host memory on a side stream); the two snapshots bracketing the current window are fused
// into one "pair record" array {a, b-a} per node that the integrator kernels gather from.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "lcs_internal.cuh"

std::atomic<int64_t> g_lcs_launches{0};
static thread_local char g_err[512] = "";

void lcs_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

// no C++ exception crosses the boundary (std::vector storage of the window plan, of the field-set keys, ...)
#define LCS_GUARD(...)                                                                           \
    try { __VA_ARGS__ } catch (const std::bad_alloc &) { lcs_set_error("host allocation failed"); return LCS_ERR_OOM; } \
    catch (...) { lcs_set_error("unexpected C++ exception"); return LCS_ERR_CUDA; }

extern "C" const char *lcs_last_error(void) { return g_err; }
extern "C" int64_t lcs_kernel_launch_count(void) { return g_lcs_launches.load(); }

// ---------------------------------------------------------------------------------------------
// pair-record build: rec[node] = { a[0..dim), 0.., (b-a)[0..dim), 0.. }   (HBM streaming, once per window)
// TV = storage type of the raw snapshot, TR = record type = the wider of storage and compute type, so that with
// fp32 data and fp64 arithmetic the difference b - a is formed in fp64 exactly as the oracle forms it.
template <int DIM, typename TV, typename TR>
__global__ void __launch_bounds__(256) build_pair_kernel(const TV *__restrict__ a, const TV *__restrict__ b,
                                                          PairRec<DIM, TR> *__restrict__ rec, int64_t nnodes)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nnodes) return;
    PairRec<DIM, TR> r;
#pragma unroll
    for (int c = 0; c < PadOf<DIM>::P; ++c) {
        TR va = (c < DIM) ? (TR)a[i * DIM + c] : TR(0);
        TR vb = (c < DIM) ? (TR)b[i * DIM + c] : TR(0);
        r.a[c] = va;
        r.d[c] = vb - va;
    }
    rec[i] = r;
}

// Cartesian grids: the record array is padded by one node per axis (np = n + 1), record (i0,i1,i2) holding node
// (i0 mod n0, i1 mod n1, i2 mod n2).  The upper corner of any cell, periodic seam included, is then at a constant
// offset from the lower one: one base address and 2^DIM constant offsets per interpolation.
template <int DIM, typename TV, typename TR>
__global__ void __launch_bounds__(256) build_pair_padded_kernel(const TV *__restrict__ a, const TV *__restrict__ b,
                                                                 PairRec<DIM, TR> *__restrict__ rec, int n0, int n1, int n2,
                                                                 int q0, int q1, int q2)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t p0 = q0, p1 = q1, p2 = q2;
    if (i >= p0 * p1 * p2) return;
    int i0 = (int)(i % p0) % n0, i1 = (int)((i / p0) % p1) % n1, i2 = (int)(i / (p0 * p1)) % n2;
    const int64_t node = i0 + (int64_t)n0 * (i1 + (int64_t)n1 * i2);
    PairRec<DIM, TR> r;
#pragma unroll
    for (int c = 0; c < PadOf<DIM>::P; ++c) {
        TR va = (c < DIM) ? (TR)a[node * DIM + c] : TR(0);
        TR vb = (c < DIM) ? (TR)b[node * DIM + c] : TR(0);
        r.a[c] = va;
        r.d[c] = vb - va;
    }
    rec[i] = r;
}

static int rec_dtype(const lcs_field *f) { return (f->vel_dtype == LCS_F64 || f->compute_dtype == LCS_F64) ? LCS_F64 : LCS_F32; }
static size_t pair_bytes(const lcs_field *f) { return (size_t)f->nrec * 2 * f->P * lcs_esize(rec_dtype(f)); }
static size_t raw_bytes(const lcs_field *f) { return (size_t)f->nnodes * f->dim * lcs_esize(f->vel_dtype); }

// Makes snapshot s resident in some raw slot (enqueueing the upload on the side stream if needed) and
// returns the slot.  `keep0/keep1` are snapshots that must not be evicted.
static lcs_status ensure_slot(lcs_field *f, int s, int keep0, int keep1, int *slot_out)
{
    if (s < 0 || s >= f->ns) { lcs_set_error("snapshot %d out of range", s); return LCS_ERR_INVALID_ARG; }
    if (!f->snap_set[s]) { lcs_set_error("snapshot %d was never set", s); return LCS_ERR_NOT_READY; }
    if (f->snap_slot[s] >= 0) { *slot_out = f->snap_slot[s]; return LCS_OK; }
    // ring mode only: pick an empty slot, else the resident snapshot farthest from s
    int best = -1, best_d = -1;
    for (int k = 0; k < f->nslots; ++k) {
        int held = f->slot_snap[k];
        if (held < 0) { best = k; break; }
        if (held == keep0 || held == keep1) continue;
        int d = abs(held - s);
        if (d > best_d) { best_d = d; best = k; }
    }
    if (best < 0) { lcs_set_error("no free snapshot slot"); return LCS_ERR_INVALID_ARG; }
    if (f->slot_snap[best] >= 0) f->snap_slot[f->slot_snap[best]] = -1;
    // do not overwrite the slot before its last reader (a pair build on the compute stream) is done
    if (f->slot_free_valid[best]) LCS_CUDA_OK(cudaStreamWaitEvent(f->side, f->slot_free[best], 0));
    LCS_CUDA_OK(cudaMemcpyAsync(f->slot[best], f->host_src[s], raw_bytes(f), cudaMemcpyHostToDevice, f->side));
    LCS_CUDA_OK(cudaEventRecord(f->slot_ready[best], f->side));
    f->info_h2d_bytes += (int64_t)raw_bytes(f);
    f->slot_snap[best] = s;
    f->snap_slot[s] = best;
    *slot_out = best;
    return LCS_OK;
}

lcs_status lcs_field_prefetch(lcs_field *f, int s, int keep0, int keep1)
{
    if (!f->ring || s < 0 || s >= f->ns || !f->snap_set[s] || f->snap_slot[s] >= 0) return LCS_OK;
    // never evict the snapshots of the window that is being integrated (keep0, keep1): the pre-blended integrator
    // reads their raw slots until the end of the window.  No other slot free => no prefetch (loaded on demand).
    int slot;
    lcs_status rc = ensure_slot(f, s, keep0, keep1, &slot);
    return rc == LCS_ERR_INVALID_ARG ? LCS_OK : rc;
}

template <int DIM, typename TV, typename TR>
static void launch_build_pair(const lcs_field *f, const void *a, const void *b, void *rec, cudaStream_t st)
{
    if (f->kind == LCS_MESH_CARTESIAN)
        LCS_LAUNCH((build_pair_padded_kernel<DIM, TV, TR>), lcs_blocks(f->nrec, 256), 256, 0, st, (const TV *)a, (const TV *)b,
                   (PairRec<DIM, TR> *)rec, f->cart.n[0], f->cart.n[1], f->cart.n[2], f->cart.np[0], f->cart.np[1], f->cart.np[2]);
    else
        LCS_LAUNCH((build_pair_kernel<DIM, TV, TR>), lcs_blocks(f->nnodes, 256), 256, 0, st, (const TV *)a, (const TV *)b,
                   (PairRec<DIM, TR> *)rec, f->nnodes);
}

lcs_status lcs_field_require_pair(lcs_field *f, int s, cudaStream_t st, const void **pair)
{
    if (s < 0 || s + 1 >= f->ns) { lcs_set_error("pair %d out of range", s); return LCS_ERR_INVALID_ARG; }
    f->pair_clock++;
    for (int k = 0; k < f->n_pair_cache; ++k)
        if (f->pair_snap[k] == s && f->pair_buf[k]) { f->pair_age[k] = f->pair_clock; *pair = f->pair_buf[k]; return LCS_OK; }
    int s0, s1;
    lcs_status rc = ensure_slot(f, s, s, s + 1, &s0);
    if (rc != LCS_OK) return rc;
    rc = ensure_slot(f, s + 1, s, s + 1, &s1);
    if (rc != LCS_OK) return rc;
    int k = 0;
    for (int j = 1; j < f->n_pair_cache; ++j)
        if (f->pair_age[j] < f->pair_age[k]) k = j;
    LCS_CUDA_OK(cudaStreamWaitEvent(st, f->slot_ready[s0], 0));
    LCS_CUDA_OK(cudaStreamWaitEvent(st, f->slot_ready[s1], 0));
    const bool v64 = f->vel_dtype == LCS_F64, r64 = rec_dtype(f) == LCS_F64;
    const void *A = f->slot[s0], *B = f->slot[s1];
    void *R = f->pair_buf[k];
    if (f->dim == 2) {
        if (v64) launch_build_pair<2, double, double>(f, A, B, R, st);
        else if (r64) launch_build_pair<2, float, double>(f, A, B, R, st);
        else launch_build_pair<2, float, float>(f, A, B, R, st);
    } else {
        if (v64) launch_build_pair<3, double, double>(f, A, B, R, st);
        else if (r64) launch_build_pair<3, float, double>(f, A, B, R, st);
        else launch_build_pair<3, float, float>(f, A, B, R, st);
    }
    LCS_CUDA_OK(cudaGetLastError());
    if (f->ring) {
        LCS_CUDA_OK(cudaEventRecord(f->slot_free[s0], st));
        LCS_CUDA_OK(cudaEventRecord(f->slot_free[s1], st));
        f->slot_free_valid[s0] = f->slot_free_valid[s1] = 1;
    }
    f->pair_snap[k] = s;
    f->pair_age[k] = f->pair_clock;
    *pair = f->pair_buf[k];
    return LCS_OK;
}

// Raw snapshots s and s + 1 for kernels that read the [node][dim] slots directly (the per-stage-time blend of the
// pre-blended integrator).  release_raw marks the end of the last reader on `st` so that the ring may reuse the slots.
lcs_status lcs_field_acquire_raw(lcs_field *f, int s, cudaStream_t st, const void **a, const void **b)
{
    if (s < 0 || s + 1 >= f->ns) { lcs_set_error("pair %d out of range", s); return LCS_ERR_INVALID_ARG; }
    int s0, s1;
    lcs_status rc = ensure_slot(f, s, s, s + 1, &s0);
    if (rc != LCS_OK) return rc;
    rc = ensure_slot(f, s + 1, s, s + 1, &s1);
    if (rc != LCS_OK) return rc;
    LCS_CUDA_OK(cudaStreamWaitEvent(st, f->slot_ready[s0], 0));
    LCS_CUDA_OK(cudaStreamWaitEvent(st, f->slot_ready[s1], 0));
    *a = f->slot[s0];
    *b = f->slot[s1];
    return LCS_OK;
}

lcs_status lcs_field_release_raw(lcs_field *f, int s, cudaStream_t st)
{
    if (!f->ring) return LCS_OK;
    for (int k = s; k <= s + 1; ++k) {
        int sl = f->snap_slot[k];
        if (sl < 0) continue;
        LCS_CUDA_OK(cudaEventRecord(f->slot_free[sl], st));
        f->slot_free_valid[sl] = 1;
    }
    return LCS_OK;
}

lcs_status lcs_scratch_check(lcs_field *f, size_t bytes)
{
    if (f->scratch.bytes >= bytes) return LCS_OK;
    lcs_set_error("the reservation (%zu bytes for %lld seeds, %lld steps) does not cover this call (%zu bytes): call lcs_field_reserve first "
                  "(the hot calls never allocate)", f->scratch.bytes, (long long)f->scratch.n_seeds, (long long)f->scratch.n_steps, bytes);
    return LCS_ERR_OOM;
}

// ---------------------------------------------------------------------------------------------
// stage-time tables, filled on the device so that lcs_advect issues no host-to-device copy.  Same operations as
// lcs_stage_tau on the host, every one rounded separately (no FMA contraction), hence the same bits.
template <typename TC>
__global__ void __launch_bounds__(128) stage_tau_kernel(double t0, double h, int64_t first, int count, double ts0, double ts1, double ts2,
                                                         double dt0, double dt1, double dt2, TC *__restrict__ tau, float *__restrict__ ftau)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const double n = (double)(first + i);
    const double ts[3] = {ts0, ts1, ts2}, dts[3] = {dt0, dt1, dt2};
    double v[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double t = __dadd_rn(t0, __dmul_rn(__dadd_rn(n, 0.5 * (double)k), h));
        v[k] = __ddiv_rn(__dsub_rn(t, ts[k]), dts[k]);
    }
    if (tau) { tau[3 * (first + i)] = (TC)v[0]; tau[3 * (first + i) + 1] = (TC)v[1]; tau[3 * (first + i) + 2] = (TC)v[2]; }
    if (ftau) {
        ftau[2 * i] = (float)v[0];
        ftau[2 * i + 1] = (float)v[1];
        if (i == count - 1) ftau[2 * count] = (float)v[2];
    }
}

lcs_status lcs_fill_stage_tau(const lcs_field *f, double t0, double h, int64_t first, int count, const int32_t s[3], void *tau,
                              float *ftau, cudaStream_t st)
{
    double ts[3], dts[3];
    for (int k = 0; k < 3; ++k) { ts[k] = f->times[s[k]]; dts[k] = f->times[s[k] + 1] - f->times[s[k]]; }
    if (f->compute_dtype == LCS_F64)
        LCS_LAUNCH((stage_tau_kernel<double>), lcs_blocks(count, 128), 128, 0, st, t0, h, first, count, ts[0], ts[1], ts[2], dts[0], dts[1], dts[2],
                   (double *)tau, ftau);
    else
        LCS_LAUNCH((stage_tau_kernel<float>), lcs_blocks(count, 128), 128, 0, st, t0, h, first, count, ts[0], ts[1], ts[2], dts[0], dts[1], dts[2],
                   (float *)tau, ftau);
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
// Window plan.  Stage times by multiplication (DESIGN reading #16): ta = t0 + n h, tb = t0 + (n+1/2) h,
// tc = t0 + (n+1) h.  The snapshot interval is that of the step's midpoint when both ends lie in it (to a
// tolerance of 1e-9 intervals: a stage time that lands on a snapshot is evaluated with tau = 1 in the
// earlier interval instead of tau = 0 in the later one -- the same value, reading #17); otherwise each
// stage time takes its own interval s = clamp(floor((t - times[0]) / dt), 0, ns-2) as the oracle does.
lcs_status lcs_plan_windows(const lcs_field *f, double t0, double h, int64_t N, std::vector<StepWindow> &windows)
{
    const double T0 = f->times[0], dt = f->dt_snap, eps = 1e-9 * dt;
    auto bracket = [&](double t) {
        double q = floor((t - T0) / dt);
        int s = q < 0.0 ? 0 : (q > (double)(f->ns - 2) ? f->ns - 2 : (int)q);
        return s;
    };
    windows.clear();
    for (int64_t n = 0; n < N; ++n) {
        double t[3] = {t0 + (double)n * h, t0 + ((double)n + 0.5) * h, t0 + ((double)n + 1.0) * h};
        int sm = bracket(t[1]);
        double lo = f->times[sm] - eps, hi = f->times[sm + 1] + eps;
        int s[3];
        if (t[0] >= lo && t[0] <= hi && t[2] >= lo && t[2] <= hi) s[0] = s[1] = s[2] = sm;
        else for (int k = 0; k < 3; ++k) s[k] = bracket(t[k]);
        if (!windows.empty()) {
            StepWindow &w = windows.back();
            if (w.s[0] == s[0] && w.s[1] == s[1] && w.s[2] == s[2] && w.count < (1 << 30)) { w.count++; continue; }
        }
        StepWindow w;
        w.first = n; w.count = 1; w.s[0] = s[0]; w.s[1] = s[1]; w.s[2] = s[2];
        windows.push_back(w);
    }
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
static lcs_status field_create_impl(const lcs_field_desc *d, lcs_field **out);
extern "C" lcs_status lcs_field_create(const lcs_field_desc *d, lcs_field **out)
{
    LCS_GUARD(return field_create_impl(d, out);)
}

static lcs_status field_create_impl(const lcs_field_desc *d, lcs_field **out)
{
    if (out) *out = nullptr;
    if (!d || !out) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    if (d->dim != 2 && d->dim != 3) { lcs_set_error("dim must be 2 or 3"); return LCS_ERR_INVALID_ARG; }
    if (d->kind != LCS_MESH_CARTESIAN && d->kind != LCS_MESH_SIMPLEX) { lcs_set_error("bad mesh kind"); return LCS_ERR_INVALID_ARG; }
    if (d->n_snapshots < 2 || !d->times) { lcs_set_error("need >= 2 snapshot times"); return LCS_ERR_INVALID_ARG; }
    if ((d->vel_dtype != LCS_F32 && d->vel_dtype != LCS_F64) || (d->compute_dtype != LCS_F32 && d->compute_dtype != LCS_F64)) {
        lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG;
    }
    if (d->max_resident_snapshots != 0 && d->max_resident_snapshots < 3) {
        lcs_set_error("max_resident_snapshots must be 0 or >= 3"); return LCS_ERR_INVALID_ARG;
    }
    double dt = d->times[1] - d->times[0];
    if (!(dt > 0)) { lcs_set_error("times must increase"); return LCS_ERR_INVALID_ARG; }
    for (int s = 1; s < d->n_snapshots; ++s)
        if (fabs((d->times[s] - d->times[s - 1]) - dt) > 1e-9 * dt) { lcs_set_error("snapshot times must be uniformly spaced"); return LCS_ERR_INVALID_ARG; }

    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) {
        lcs_set_error("no CUDA device: liblcs has no CPU fallback");
        return LCS_ERR_CUDA;
    }
    lcs_field *f = new (std::nothrow) lcs_field();
    if (!f) return LCS_ERR_OOM;
    f->dim = d->dim; f->kind = d->kind; f->vel_dtype = d->vel_dtype; f->compute_dtype = d->compute_dtype;
    f->P = (d->dim == 2) ? 2 : 4;
    f->times.assign(d->times, d->times + d->n_snapshots);
    f->dt_snap = dt;
    f->ns = d->n_snapshots;
    lcs_status rc = LCS_OK;
    if (d->kind == LCS_MESH_CARTESIAN) {
        int64_t nn = 1;
        for (int a = 0; a < 3; ++a) {
            int32_t na = (a < d->dim) ? d->n[a] : 1;
            if (a < d->dim && (na < 2 || !(d->spacing[a] > 0))) { lcs_set_error("bad Cartesian grid on axis %d", a); delete f; return LCS_ERR_INVALID_ARG; }
            f->cart.n[a] = na;
            f->cart.periodic[a] = (a < d->dim) ? (d->periodic[a] != 0) : 0;
            f->cart.pow2[a] = (na & (na - 1)) == 0;
            f->cart.origin[a] = (a < d->dim) ? d->origin[a] : 0.0;
            f->cart.spacing[a] = (a < d->dim) ? d->spacing[a] : 1.0;
            f->cart.inv[a] = 1.0 / f->cart.spacing[a];
            nn *= na;
        }
        if (nn >= (1LL << 31)) { lcs_set_error("grid too large for int32 node ids"); delete f; return LCS_ERR_INVALID_ARG; }
        f->nnodes = nn;
        f->nrec = 1;
        for (int a = 0; a < 3; ++a) {
            f->cart.np[a] = a < d->dim ? d->n[a] + 1 : 1;
            f->nrec *= (int64_t)f->cart.np[a];
        }
        if (f->nrec >= (1LL << 31)) { lcs_set_error("grid too large for int32 node ids"); delete f; return LCS_ERR_INVALID_ARG; }
    } else {
        if (d->n_vertices < d->dim + 1 || d->n_cells < 1 || !d->vertices || !d->cells || d->n_vertices >= (1LL << 31) ||
            d->n_cells >= (1LL << 31) / (d->dim + 1)) {
            lcs_set_error("bad simplex mesh sizes / null pointers"); delete f; return LCS_ERR_INVALID_ARG;
        }
        f->nnodes = d->n_vertices;
        f->nrec = d->n_vertices;
        f->mesh.nv = d->n_vertices; f->mesh.nc = d->n_cells;
        rc = lcs_simplex_build(f, d->vertices, d->cells);
        if (rc != LCS_OK) { lcs_field_destroy(f); return rc; }
    }
    f->ring = d->max_resident_snapshots != 0 && d->max_resident_snapshots < d->n_snapshots;
    f->nslots = f->ring ? d->max_resident_snapshots : d->n_snapshots;
    f->slot.assign(f->nslots, nullptr);
    f->slot_snap.assign(f->nslots, -1);
    f->slot_ready.assign(f->nslots, nullptr);
    f->slot_free.assign(f->nslots, nullptr);
    f->slot_free_valid.assign(f->nslots, 0);
    f->snap_slot.assign(f->ns, -1);
    f->snap_set.assign(f->ns, 0);
    f->host_src.assign(f->ns, nullptr);
    cudaError_t e = cudaStreamCreateWithFlags(&f->side, cudaStreamNonBlocking);
    for (int k = 0; k < f->nslots && e == cudaSuccess; ++k) {
        e = cudaEventCreateWithFlags(&f->slot_ready[k], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->slot_free[k], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) { lcs_set_error("stream/event creation failed: %s", cudaGetErrorString(e)); lcs_field_destroy(f); return LCS_ERR_CUDA; }
    // the snapshot window and the pair-record cache are allocated here, once: the hot calls never allocate
    for (int k = 0; k < f->nslots && e == cudaSuccess; ++k) e = cudaMalloc(&f->slot[k], raw_bytes(f));
    if (!f->ring && f->ns - 1 <= lcs_field::kMaxPairCache && (size_t)(f->ns - 1) * pair_bytes(f) <= ((size_t)256 << 20)) f->n_pair_cache = f->ns - 1 > 4 ? f->ns - 1 : 4;
    for (int k = 0; k < f->n_pair_cache && e == cudaSuccess; ++k) e = cudaMalloc(&f->pair_buf[k], pair_bytes(f));
    if (e != cudaSuccess) {
        lcs_set_error("allocating the snapshot window failed: %s", cudaGetErrorString(e));
        lcs_field_destroy(f);
        return e == cudaErrorMemoryAllocation ? LCS_ERR_OOM : LCS_ERR_CUDA;
    }
    *out = f;
    return LCS_OK;
}

extern "C" void lcs_field_destroy(lcs_field *f)
{
    if (!f) return;
    cudaDeviceSynchronize();
    for (void *p : f->slot) if (p) cudaFree(p);
    for (cudaEvent_t ev : f->slot_ready) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : f->slot_free) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : f->win_ev) cudaEventDestroy(ev);
    for (int k = 0; k < f->n_pair_cache; ++k) if (f->pair_buf[k]) cudaFree(f->pair_buf[k]);
    if (f->scratch.buf) cudaFree(f->scratch.buf);
    for (FieldSet &fs : f->field_sets) if (fs.buf) cudaFree(fs.buf);
    if (f->h_seeds) cudaFree(f->h_seeds);
    if (f->h_flow) cudaFree(f->h_flow);
    if (f->h_ftle) cudaFree(f->h_ftle);
    if (f->h_flag) cudaFree(f->h_flag);
    if (f->h_cg) cudaFree(f->h_cg);
    if (f->h_step) cudaFree(f->h_step);
    if (f->hs_flow) cudaFree(f->hs_flow);
    if (f->hs_ftle) cudaFree(f->hs_ftle);
    if (f->hs_cg) cudaFree(f->hs_cg);
    if (f->hs_flag) cudaFree(f->hs_flag);
    if (f->hs_step) cudaFree(f->hs_step);
    lcs_simplex_free(f);
    if (f->side) cudaStreamDestroy(f->side);
    delete f;
}

extern "C" lcs_status lcs_field_set_snapshot(lcs_field *f, int32_t s, const void *vel, int32_t is_device_ptr)
{
    if (!f || !vel) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    if (s < 0 || s >= f->ns) { lcs_set_error("snapshot index %d out of range", s); return LCS_ERR_INVALID_ARG; }
    // any cached pair built from the old contents is stale
    for (int k = 0; k < f->n_pair_cache; ++k)
        if (f->pair_snap[k] == s || f->pair_snap[k] == s - 1) f->pair_snap[k] = -1;
    for (FieldSet &fs : f->field_sets)
        if (fs.pair == s || fs.pair == s - 1) { fs.pair = -1; fs.tau.clear(); }
    if (f->ring) {
        if (is_device_ptr) { lcs_set_error("ring mode streams snapshots from HOST memory"); return LCS_ERR_INVALID_ARG; }
        f->host_src[s] = vel;
        f->snap_set[s] = 1;
        if (f->snap_slot[s] >= 0) { f->slot_snap[f->snap_slot[s]] = -1; f->snap_slot[s] = -1; }
        return LCS_OK;
    }
    LCS_CUDA_OK(cudaMemcpyAsync(f->slot[s], vel, raw_bytes(f), is_device_ptr ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, f->side));
    LCS_CUDA_OK(cudaEventRecord(f->slot_ready[s], f->side));
    if (!is_device_ptr) f->info_h2d_bytes += (int64_t)raw_bytes(f);
    f->slot_snap[s] = s;
    f->snap_slot[s] = s;
    f->snap_set[s] = 1;
    return LCS_OK;
}

extern "C" lcs_status lcs_field_sync(lcs_field *f)
{
    if (!f) { lcs_set_error("null field"); return LCS_ERR_INVALID_ARG; }
    LCS_CUDA_OK(cudaStreamSynchronize(f->side));
    return LCS_OK;
}

extern "C" lcs_status lcs_field_set_option(lcs_field *f, const char *key, int64_t value)
{
    if (!f || !key) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    if (!strcmp(key, "integrator") && value >= 0 && value <= 3) f->opt_integrator = value;
    else if (!strcmp(key, "bundle") && value >= -1 && value <= 1) f->opt_bundle = value;
    else if (!strcmp(key, "bundle_steps") && value >= 0) f->opt_bundle_steps = value;
    else if (!strcmp(key, "bundle_order") && value >= -1 && value <= 3) f->opt_bundle_order = value;
    else if (!strcmp(key, "simplex_order") && (value == 0 || value == 1)) f->opt_simplex_order = value;
    else if (!strcmp(key, "tma") && value >= 0 && value <= 2) f->opt_tma = value;
    else if (!strcmp(key, "tma_cap") && value >= 64 && value <= 3500) {
        f->opt_tma_cap = value;
        lcs_status rc = lcs_cart_tma_configure(f);
        if (rc != LCS_OK) return rc;
    }
    else if (!strcmp(key, "ld256") && (value == 0 || value == 1)) f->opt_ld256 = value;
    else if (!strcmp(key, "preblend") && value >= -1 && value <= 1) f->opt_preblend = value;
    else if (!strcmp(key, "field_sets") && value >= 0 && value <= 64) {      // set-up: the next lcs_field_reserve allocates the sets
        f->opt_field_sets = value;
        cudaDeviceSynchronize();
        for (FieldSet &fs : f->field_sets) if (fs.buf) cudaFree(fs.buf);
        f->field_sets.clear();
    }
    else if (!strcmp(key, "field_sets_clear")) { for (FieldSet &fs : f->field_sets) { fs.pair = -1; fs.tau.clear(); } }
    else if (!strcmp(key, "preblend_steps") && value >= 1 && value <= 256) f->opt_preblend_steps = value;
    else if (!strcmp(key, "time_windows") && (value == 0 || value == 1)) { f->opt_time_windows = value; f->win_ev_used = 0; }
    else if (!strcmp(key, "block") && (value == 0 || (value >= 32 && value <= 1024 && value % 32 == 0))) f->opt_block = value;
    else { lcs_set_error("unknown option or bad value: %s=%lld", key, (long long)value); return LCS_ERR_INVALID_ARG; }
    return LCS_OK;
}

static lcs_status field_get_info_impl(const lcs_field *f, const char *key, int64_t *value);
extern "C" lcs_status lcs_field_get_info(const lcs_field *f, const char *key, int64_t *value)
{
    LCS_GUARD(return field_get_info_impl(f, key, value);)
}

static lcs_status field_get_info_impl(const lcs_field *f, const char *key, int64_t *value)
{
    if (!f || !key || !value) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    if (!strcmp(key, "windows")) *value = f->info_windows;
    else if (!strcmp(key, "series_layers")) *value = f->info_series_layers;
    else if (!strcmp(key, "h2d_bytes")) *value = f->info_h2d_bytes;
    else if (!strcmp(key, "n_nodes")) *value = f->nnodes;
    else if (!strcmp(key, "n_cells")) *value = f->kind == LCS_MESH_SIMPLEX ? f->mesh.nc : 0;
    else if (!strcmp(key, "n_bins")) *value = f->kind == LCS_MESH_SIMPLEX ? (int64_t)f->mesh.nb[0] * f->mesh.nb[1] * f->mesh.nb[2] : 0;
    else if (!strcmp(key, "ring")) *value = f->ring;
    else if (!strcmp(key, "field_set_hits")) *value = f->info_field_set_hits;
    else if (!strcmp(key, "field_set_misses")) *value = f->info_field_set_misses;
    else if (!strcmp(key, "window_launches")) *value = (int64_t)(f->win_ev_used / 2);
    else if (!strcmp(key, "window_time_ns")) {          // synchronises; sum of the bracketed launch durations
        double ms = 0.0;
        for (size_t k = 0; k + 1 < f->win_ev_used; k += 2) {
            float e = 0.f;
            if (cudaEventSynchronize(f->win_ev[k + 1]) != cudaSuccess || cudaEventElapsedTime(&e, f->win_ev[k], f->win_ev[k + 1]) != cudaSuccess) {
                lcs_set_error("window timing events not complete"); return LCS_ERR_CUDA;
            }
            ms += e;
        }
        *value = (int64_t)(ms * 1e6);
    }
    else if (!strcmp(key, "locate_fallbacks") || !strcmp(key, "locate_hops") || !strcmp(key, "locate_max_hops") || !strcmp(key, "locate_random_walks") ||
             !strcmp(key, "walk_cap_hits") || !strcmp(key, "walk_fallbacks")) {
        *value = 0;
        if (f->kind == LCS_MESH_SIMPLEX) {
            unsigned long long h[16] = {0};
            cudaMemcpy(h, f->mesh.stats, sizeof h, cudaMemcpyDeviceToHost);
            // fallbacks of the in-advect re-locations ([8], [11]) count as locate fallbacks / random walks too
            if (!strcmp(key, "locate_fallbacks")) *value = (int64_t)(h[0] + h[8]);
            else if (!strcmp(key, "locate_hops")) *value = (int64_t)h[1];
            else if (!strcmp(key, "locate_max_hops")) *value = (int64_t)h[2];
            else if (!strcmp(key, "locate_random_walks")) *value = (int64_t)(h[3] + h[11]);
            else if (!strcmp(key, "walk_cap_hits")) *value = (int64_t)h[4];
            else *value = (int64_t)h[5];
        }
    }
    else if (!strcmp(key, "scratch_bytes")) *value = (int64_t)f->scratch.bytes;
    else if (!strcmp(key, "n_boundary_faces")) {
        *value = 0;
        if (f->kind == LCS_MESH_SIMPLEX) {
            std::vector<int32_t> nb((size_t)f->mesh.nc * (f->dim + 1));
            cudaMemcpy(nb.data(), f->mesh.neigh, nb.size() * 4, cudaMemcpyDeviceToHost);
            int64_t c = 0;
            for (int32_t v : nb) c += (v < 0);
            *value = c;
        }
    } else { lcs_set_error("unknown info key %s", key); return LCS_ERR_INVALID_ARG; }
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" lcs_status lcs_locate(lcs_field *f, int64_t n, const double *pos, int32_t *cell, double *bary, void *cuda_stream)
{
    if (!f || n < 0 || (n > 0 && (!pos || !cell))) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    if (n == 0) return LCS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return f->kind == LCS_MESH_CARTESIAN ? lcs_cart_locate(f, n, pos, cell, bary, st) : lcs_simplex_locate(f, n, pos, cell, bary, st);
}

static lcs_status check_interval(const lcs_field *f, double t0, double tf, double h, int64_t *N)
{
    if (!(h != 0.0) || !isfinite(h) || !isfinite(t0) || !isfinite(tf)) { lcs_set_error("h must be finite and non-zero"); return LCS_ERR_INVALID_ARG; }
    double T = tf - t0;
    if (T == 0.0 || (T > 0) != (h > 0)) { lcs_set_error("sign(h) must equal sign(tf - t0)"); return LCS_ERR_INVALID_ARG; }
    int64_t n = llround(T / h);
    if (n < 1 || fabs((double)n * h - T) > 1e-9 * fabs(T)) { lcs_set_error("(tf-t0)/h must be a positive integer (no partial last step)"); return LCS_ERR_INVALID_ARG; }
    if (n >= (1LL << 24)) { lcs_set_error("more than 2^24 - 1 steps per call: split the interval (the flow map of one call seeds the next)"); return LCS_ERR_INVALID_ARG; }
    double eps = 1e-9 * f->dt_snap, lo = f->times.front() - eps, hi = f->times.back() + eps;
    if (t0 < lo || t0 > hi || tf < lo || tf > hi) { lcs_set_error("[t0,tf] = [%g,%g] outside the snapshot times [%g,%g]", t0, tf, f->times.front(), f->times.back()); return LCS_ERR_TIME_RANGE; }
    *N = n;
    return LCS_OK;
}

extern "C" lcs_status lcs_field_reserve(lcs_field *f, int64_t n_seeds, int64_t n_steps)
{
    if (!f) { lcs_set_error("null field"); return LCS_ERR_INVALID_ARG; }
    if (n_seeds < 1 || n_steps < 1 || n_seeds >= (1LL << 31) || n_steps >= (1LL << 24)) {
        lcs_set_error("lcs_field_reserve: need 1 <= n_seeds < 2^31 and 1 <= n_steps < 2^24"); return LCS_ERR_INVALID_ARG;
    }
    LCS_GUARD(
        const size_t need = f->kind == LCS_MESH_CARTESIAN ? lcs_cart_scratch_bytes(f, n_seeds, n_steps) : lcs_simplex_scratch_bytes(f, n_seeds, n_steps);
        if (need > f->scratch.bytes) {
            if (f->scratch.buf) { cudaDeviceSynchronize(); cudaFree(f->scratch.buf); f->scratch.buf = nullptr; f->scratch.bytes = 0; }
            LCS_CUDA_OK(cudaMalloc(&f->scratch.buf, need));
            f->scratch.bytes = need;
        }
        if (n_seeds > f->scratch.n_seeds) f->scratch.n_seeds = n_seeds;
        if (n_steps > f->scratch.n_steps) f->scratch.n_steps = n_steps;
        // resident sets of blended fields (option "field_sets"): all of them, now
        const size_t set_bytes = f->kind == LCS_MESH_CARTESIAN ? lcs_cart_field_set_bytes(f, n_steps) : 0;
        if (f->opt_field_sets > 0 && set_bytes > 0) {
            f->field_sets.resize((size_t)f->opt_field_sets);
            for (FieldSet &fs : f->field_sets) {
                if (fs.bytes >= set_bytes) continue;
                fs.pair = -1; fs.tau.clear();
                if (fs.buf) { cudaDeviceSynchronize(); cudaFree(fs.buf); fs.buf = nullptr; fs.bytes = 0; }
                LCS_CUDA_OK(cudaMalloc(&fs.buf, set_bytes));
                fs.bytes = set_bytes;
            }
        }
        return LCS_OK;
    )
}

extern "C" lcs_status lcs_advect(lcs_field *f, int64_t n, const void *seeds, double t0, double tf, double h, void *flowmap,
                                 uint8_t *exit_flag, int32_t *exit_step, void *cuda_stream)
{
    if (!f || n < 0 || (n > 0 && (!seeds || !flowmap))) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    int64_t N = 0;
    lcs_status rc = check_interval(f, t0, tf, h, &N);
    if (rc != LCS_OK) return rc;
    if (n == 0) return LCS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LCS_GUARD(
        return f->kind == LCS_MESH_CARTESIAN ? lcs_cart_advect(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st)
                                             : lcs_simplex_advect(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    )
}

// ---------------------------------------------------------------------------------------------
static lcs_status series_args(lcs_field *f, int64_t n, int32_t n_vol, const double *t_start, double T, double h, int64_t *N)
{
    if (!f || n < 1 || n_vol < 1 || !t_start) { lcs_set_error("null argument, n < 1 or n_vol < 1"); return LCS_ERR_INVALID_ARG; }
    if (n_vol > 65536 || (int64_t)n_vol * n >= (1LL << 31)) { lcs_set_error("n_vol * n must stay below 2^31"); return LCS_ERR_INVALID_ARG; }
    int64_t Nk = 0;
    for (int k = 0; k < n_vol; ++k) {
        lcs_status rc = check_interval(f, t_start[k], t_start[k] + T, h, &Nk);
        if (rc != LCS_OK) return rc;
        if (k > 0 && Nk != *N) { lcs_set_error("volumes of a series take the same number of steps"); return LCS_ERR_INVALID_ARG; }
        *N = Nk;
    }
    return LCS_OK;
}

extern "C" lcs_status lcs_advect_series_reserve(lcs_field *f, int64_t n, int32_t n_vol, const double *t_start, double T, double h)
{
    int64_t N = 0;
    lcs_status rc = series_args(f, n, n_vol, t_start, T, h, &N);
    if (rc != LCS_OK) return rc;
    LCS_GUARD(
        int64_t cap = n;
        if (f->kind == LCS_MESH_CARTESIAN) {
            rc = lcs_cart_advect_series(f, n, nullptr, n_vol, t_start, h, N, nullptr, nullptr, nullptr, nullptr, &cap);
            if (rc != LCS_OK) return rc;
        }
        return lcs_field_reserve(f, cap, N);
    )
}

extern "C" lcs_status lcs_advect_series(lcs_field *f, int64_t n, const void *seeds, int32_t n_vol, const double *t_start, double T, double h,
                                        void *flowmaps, uint8_t *exit_flags, int32_t *exit_steps, void *cuda_stream)
{
    int64_t N = 0;
    lcs_status rc = series_args(f, n, n_vol, t_start, T, h, &N);
    if (rc != LCS_OK) return rc;
    if (!seeds || !flowmaps) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LCS_GUARD(
        if (f->kind == LCS_MESH_CARTESIAN)
            return lcs_cart_advect_series(f, n, seeds, n_vol, t_start, h, N, flowmaps, exit_flags, exit_steps, st, nullptr);
        const size_t es = lcs_esize(f->compute_dtype);
        for (int k = 0; k < n_vol; ++k) {
            rc = lcs_simplex_advect(f, n, seeds, t_start[k], h, N, (char *)flowmaps + (size_t)k * n * f->dim * es,
                                    exit_flags ? exit_flags + (size_t)k * n : nullptr, exit_steps ? exit_steps + (size_t)k * n : nullptr, st);
            if (rc != LCS_OK) return rc;
        }
        return LCS_OK;
    )
}

// ---------------------------------------------------------------------------------------------
extern "C" lcs_status lcs_ftle_host(lcs_field *f, const int32_t ng[3], const double seed_spacing[3], const int32_t seed_periodic[3],
                                    const double period[3], const void *seeds_host, double t0, double tf, double h,
                                    void *flowmap_host, uint8_t *exit_flag_host, int32_t *exit_step_host, void *cg_host, void *ftle_host)
{
    if (!f || !ng || !seeds_host || !ftle_host) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    int64_t n = (int64_t)ng[0] * ng[1] * (f->dim == 3 ? ng[2] : 1);
    if (n <= 0) { lcs_set_error("empty seed grid"); return LCS_ERR_INVALID_ARG; }
    int64_t N = 0;
    lcs_status rc = check_interval(f, t0, tf, h, &N);
    if (rc != LCS_OK) return rc;
    rc = lcs_field_reserve(f, n, N);                       // this convenience call is synchronous set-up + run
    if (rc != LCS_OK) return rc;
    const size_t es = lcs_esize(f->compute_dtype), ncg = f->dim == 2 ? 3 : 6;
    if (f->h_cap < n || (cg_host && !f->h_cg) || (exit_step_host && !f->h_step)) {
        cudaDeviceSynchronize();
        if (f->h_seeds) cudaFree(f->h_seeds);
        if (f->h_ftle) cudaFree(f->h_ftle);
        if (f->h_flag) cudaFree(f->h_flag);
        if (f->h_cg) cudaFree(f->h_cg);
        if (f->h_step) cudaFree(f->h_step);
        f->h_seeds = f->h_ftle = f->h_cg = nullptr; f->h_flag = nullptr; f->h_step = nullptr;
        const int64_t cap = n > f->h_cap ? n : f->h_cap;
        f->h_cap = 0;
        LCS_CUDA_OK(cudaMalloc(&f->h_seeds, (size_t)cap * f->dim * es));
        LCS_CUDA_OK(cudaMalloc(&f->h_ftle, (size_t)cap * es));
        LCS_CUDA_OK(cudaMalloc((void **)&f->h_flag, (size_t)cap));
        if (cg_host) LCS_CUDA_OK(cudaMalloc(&f->h_cg, (size_t)cap * ncg * es));
        if (exit_step_host) LCS_CUDA_OK(cudaMalloc((void **)&f->h_step, (size_t)cap * 4));
        f->h_cap = cap;
    }
    cudaStream_t st = 0;
    LCS_CUDA_OK(cudaMemcpyAsync(f->h_seeds, seeds_host, (size_t)n * f->dim * es, cudaMemcpyHostToDevice, st));
    rc = lcs_advect(f, n, f->h_seeds, t0, tf, h, f->h_seeds, f->h_flag, exit_step_host ? f->h_step : nullptr, st);   // flow map in place
    if (rc != LCS_OK) return rc;
    rc = lcs_cg_ftle(f->dim, f->compute_dtype, ng, seed_spacing, seed_periodic, period, f->h_seeds, f->h_flag, tf - t0,
                     cg_host ? f->h_cg : nullptr, f->h_ftle, nullptr, st);
    if (rc != LCS_OK) return rc;
    LCS_CUDA_OK(cudaMemcpyAsync(ftle_host, f->h_ftle, (size_t)n * es, cudaMemcpyDeviceToHost, st));
    if (cg_host) LCS_CUDA_OK(cudaMemcpyAsync(cg_host, f->h_cg, (size_t)n * ncg * es, cudaMemcpyDeviceToHost, st));
    if (flowmap_host) LCS_CUDA_OK(cudaMemcpyAsync(flowmap_host, f->h_seeds, (size_t)n * f->dim * es, cudaMemcpyDeviceToHost, st));
    if (exit_flag_host) LCS_CUDA_OK(cudaMemcpyAsync(exit_flag_host, f->h_flag, (size_t)n, cudaMemcpyDeviceToHost, st));
    if (exit_step_host) LCS_CUDA_OK(cudaMemcpyAsync(exit_step_host, f->h_step, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    LCS_CUDA_OK(cudaStreamSynchronize(st));
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" lcs_status lcs_ftle_series_host(lcs_field *f, const int32_t ng[3], const double seed_spacing[3], const int32_t seed_periodic[3],
                                           const double period[3], const void *seeds_host, int32_t n_vol, const double *t_start, double T, double h,
                                           void *flowmaps_host, uint8_t *exit_flags_host, int32_t *exit_steps_host, void *cg_host, void *ftle_host)
{
    if (!f || !ng || !seeds_host || !ftle_host || !t_start || n_vol < 1) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    const int64_t n = (int64_t)ng[0] * ng[1] * (f->dim == 3 ? ng[2] : 1);
    if (n <= 0) { lcs_set_error("empty seed grid"); return LCS_ERR_INVALID_ARG; }
    lcs_status rc = lcs_advect_series_reserve(f, n, n_vol, t_start, T, h);      // this convenience call is synchronous set-up + run
    if (rc != LCS_OK) return rc;
    const size_t es = lcs_esize(f->compute_dtype), ncg = f->dim == 2 ? 3 : 6;
    const int64_t tot = n * n_vol;
    if (f->h_cap < n) {                                      // seeds staging shared with lcs_ftle_host
        cudaDeviceSynchronize();
        if (f->h_seeds) cudaFree(f->h_seeds);
        if (f->h_ftle) cudaFree(f->h_ftle);
        if (f->h_flag) cudaFree(f->h_flag);
        if (f->h_cg) cudaFree(f->h_cg);
        if (f->h_step) cudaFree(f->h_step);
        f->h_seeds = f->h_ftle = f->h_cg = nullptr; f->h_flag = nullptr; f->h_step = nullptr; f->h_cap = 0;
        LCS_CUDA_OK(cudaMalloc(&f->h_seeds, (size_t)n * f->dim * es));
        LCS_CUDA_OK(cudaMalloc(&f->h_ftle, (size_t)n * es));
        LCS_CUDA_OK(cudaMalloc((void **)&f->h_flag, (size_t)n));
        f->h_cap = n;
    }
    if (f->hs_cap < tot || (cg_host && !f->hs_cg)) {
        cudaDeviceSynchronize();
        if (f->hs_flow) cudaFree(f->hs_flow);
        if (f->hs_ftle) cudaFree(f->hs_ftle);
        if (f->hs_cg) cudaFree(f->hs_cg);
        if (f->hs_flag) cudaFree(f->hs_flag);
        if (f->hs_step) cudaFree(f->hs_step);
        f->hs_flow = f->hs_ftle = f->hs_cg = nullptr; f->hs_flag = nullptr; f->hs_step = nullptr;
        const int64_t cap = tot > f->hs_cap ? tot : f->hs_cap;
        f->hs_cap = 0;
        LCS_CUDA_OK(cudaMalloc(&f->hs_flow, (size_t)cap * f->dim * es));
        LCS_CUDA_OK(cudaMalloc(&f->hs_ftle, (size_t)cap * es));
        LCS_CUDA_OK(cudaMalloc((void **)&f->hs_flag, (size_t)cap));
        LCS_CUDA_OK(cudaMalloc((void **)&f->hs_step, (size_t)cap * 4));
        if (cg_host) LCS_CUDA_OK(cudaMalloc(&f->hs_cg, (size_t)cap * ncg * es));
        f->hs_cap = cap;
    }
    cudaStream_t st = 0;
    LCS_CUDA_OK(cudaMemcpyAsync(f->h_seeds, seeds_host, (size_t)n * f->dim * es, cudaMemcpyHostToDevice, st));
    rc = lcs_advect_series(f, n, f->h_seeds, n_vol, t_start, T, h, f->hs_flow, f->hs_flag, f->hs_step, st);
    if (rc != LCS_OK) return rc;
    for (int k = 0; k < n_vol; ++k) {
        rc = lcs_cg_ftle(f->dim, f->compute_dtype, ng, seed_spacing, seed_periodic, period, (char *)f->hs_flow + (size_t)k * n * f->dim * es,
                         f->hs_flag + (size_t)k * n, T, cg_host ? (char *)f->hs_cg + (size_t)k * n * ncg * es : nullptr,
                         (char *)f->hs_ftle + (size_t)k * n * es, nullptr, st);
        if (rc != LCS_OK) return rc;
    }
    LCS_CUDA_OK(cudaMemcpyAsync(ftle_host, f->hs_ftle, (size_t)tot * es, cudaMemcpyDeviceToHost, st));
    if (cg_host) LCS_CUDA_OK(cudaMemcpyAsync(cg_host, f->hs_cg, (size_t)tot * ncg * es, cudaMemcpyDeviceToHost, st));
    if (flowmaps_host) LCS_CUDA_OK(cudaMemcpyAsync(flowmaps_host, f->hs_flow, (size_t)tot * f->dim * es, cudaMemcpyDeviceToHost, st));
    if (exit_flags_host) LCS_CUDA_OK(cudaMemcpyAsync(exit_flags_host, f->hs_flag, (size_t)tot, cudaMemcpyDeviceToHost, st));
    if (exit_steps_host) LCS_CUDA_OK(cudaMemcpyAsync(exit_steps_host, f->hs_step, (size_t)tot * 4, cudaMemcpyDeviceToHost, st));
    LCS_CUDA_OK(cudaStreamSynchronize(st));
    return LCS_OK;
}
