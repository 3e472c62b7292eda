// simplex.cu -- triangle / tetrahedral meshes: device-built face adjacency and uniform bin grid, cell
// search by walking (row a2), barycentric space + linear time interpolation (row a3) and the RK4
// integrator (row a4), for sm_100a.
//
// Paper: "an efficient local cell search strategy for unstructured grids [27] ... designed for
// tetrahedral grids (or triangular grids in 2D)"; the Seed filter "computes which cell in
// the velocity field mesh each seed point is located in"; the cell search "readily
// facilitates spatial interpolation" through its natural coordinates; each of the four RK4
// evaluations needs a preceding cell search.
//
// Two predicates are used on purpose:
//  * lcs_locate and the seeds' initial cells use the CANONICAL fp64 face predicate (face vertices sorted by
//    id, every product/sum rounded separately, ties as if the point were p + (eps, eps^2, eps^3)), which
//    makes the owner of a point unique and bit-reproducible;
//  * the walk inside the integrator uses precomputed per-cell affine maps lambda = M (p - v0) in the compute
//    dtype with a small tolerance.  P1 interpolation is continuous across faces, so a different-but-adjacent
//    cell changes the velocity at rounding level only.
#include <math.h>

#include <algorithm>
#include <cub/cub.cuh>

#include "bundle_sort.cuh"
#include "lcs_internal.cuh"

namespace {

// ---------------------------------------------------------------------------------------------
// canonical predicate (must match oracle/lcs_oracle.c face_side bit for bit: no FMA contraction)
template <int DIM> __device__ __forceinline__ void sort_ids(int32_t *v)
{
    if (v[0] > v[1]) { int32_t t = v[0]; v[0] = v[1]; v[1] = t; }
    if constexpr (DIM == 3) {
        if (v[1] > v[2]) { int32_t t = v[1]; v[1] = v[2]; v[2] = t; }
        if (v[0] > v[1]) { int32_t t = v[0]; v[0] = v[1]; v[1] = t; }
    }
}

template <int DIM> __device__ __forceinline__ void face_ids(const int32_t *__restrict__ cells, int64_t c, int j, int32_t *fv)
{
    int k = 0;
#pragma unroll
    for (int i = 0; i <= DIM; ++i)
        if (i != j) fv[k++] = cells[c * (DIM + 1) + i];
    sort_ids<DIM>(fv);
}

template <int DIM>
__device__ __forceinline__ bool face_side(const double *__restrict__ verts, const int32_t *fv, const double *p, bool *strict = nullptr)
{
    if constexpr (DIM == 2) {
        const double *a = verts + 2 * (int64_t)fv[0], *b = verts + 2 * (int64_t)fv[1];
        double ax = a[0], ay = a[1];
        double ex = __dsub_rn(b[0], ax), ey = __dsub_rn(b[1], ay);
        double s = __dsub_rn(__dmul_rn(ex, __dsub_rn(p[1], ay)), __dmul_rn(ey, __dsub_rn(p[0], ax)));
        if (strict) *strict = s != 0.0;
        if (s != 0.0) return s > 0.0;
        if (ey != 0.0) return -ey > 0.0;
        return ex > 0.0;
    } else {
        const double *a = verts + 3 * (int64_t)fv[0], *b = verts + 3 * (int64_t)fv[1], *c = verts + 3 * (int64_t)fv[2];
        double ax = a[0], ay = a[1], az = a[2];
        double ux = __dsub_rn(b[0], ax), uy = __dsub_rn(b[1], ay), uz = __dsub_rn(b[2], az);
        double vx = __dsub_rn(c[0], ax), vy = __dsub_rn(c[1], ay), vz = __dsub_rn(c[2], az);
        double nx = __dsub_rn(__dmul_rn(uy, vz), __dmul_rn(uz, vy));
        double ny = __dsub_rn(__dmul_rn(uz, vx), __dmul_rn(ux, vz));
        double nz = __dsub_rn(__dmul_rn(ux, vy), __dmul_rn(uy, vx));
        double wx = __dsub_rn(p[0], ax), wy = __dsub_rn(p[1], ay), wz = __dsub_rn(p[2], az);
        double s = __dadd_rn(__dadd_rn(__dmul_rn(nx, wx), __dmul_rn(ny, wy)), __dmul_rn(nz, wz));
        if (strict) *strict = s != 0.0;
        if (s != 0.0) return s > 0.0;
        if (nx != 0.0) return nx > 0.0;
        if (ny != 0.0) return ny > 0.0;
        return nz > 0.0;
    }
}

// first face (local order) whose canonical side test fails for p, or -1 if cell c owns p
template <int DIM>
__device__ __forceinline__ int first_failing_face(const double *__restrict__ verts, const int32_t *__restrict__ cells,
                                                  const uint8_t *__restrict__ oppside, int64_t c, const double *p)
{
    const unsigned opp = oppside[c];
#pragma unroll
    for (int j = 0; j <= DIM; ++j) {
        int32_t fv[DIM];
        face_ids<DIM>(cells, c, j, fv);
        bool sp = face_side<DIM>(verts, fv, p);
        if (sp != (bool)((opp >> j) & 1u)) return j;
    }
    return -1;
}

// The walk's view of cell c: first failing face (local order, -1 = c owns p) and whether p lies STRICTLY beyond a hull
// face of c.  The meshes are triangulations of convex hulls (Delaunay), so a point strictly beyond a hull face is in
// no cell: the walk stops there instead of circling along the hull, where Qhull's near-flat boundary slivers are not
// numerically Delaunay and the visibility walk can cycle.  (A point exactly ON a hull plane is left to the
// first-failing-face rule, so ties resolve exactly as in the oracle.)
template <int DIM>
__device__ __forceinline__ int walk_probe(const double *__restrict__ verts, const int32_t *__restrict__ cells,
                                          const int32_t *__restrict__ neigh, const uint8_t *__restrict__ oppside, int64_t c,
                                          const double *p, bool *beyond_hull)
{
    const unsigned opp = oppside[c];
    int first = -1;
    bool out = false;
#pragma unroll
    for (int j = 0; j <= DIM; ++j) {
        int32_t fv[DIM];
        face_ids<DIM>(cells, c, j, fv);
        bool strict;
        bool sp = face_side<DIM>(verts, fv, p, &strict);
        if (sp != (bool)((opp >> j) & 1u)) {
            if (first < 0) first = j;
            if (strict && neigh[c * (DIM + 1) + j] < 0) out = true;
        }
    }
    *beyond_hull = out;
    return first;
}

// ---------------------------------------------------------------------------------------------
// create-time kernels
template <int DIM>
__global__ void __launch_bounds__(256) face_key_kernel(const int32_t *__restrict__ cells, int64_t nfaces,
                                                        uint64_t *__restrict__ key_hi, uint32_t *__restrict__ key_lo,
                                                        int32_t *__restrict__ face_id)
{
    int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= nfaces) return;
    int32_t fv[DIM];
    face_ids<DIM>(cells, f / (DIM + 1), (int)(f % (DIM + 1)), fv);
    key_hi[f] = ((uint64_t)(uint32_t)fv[0] << 32) | (uint32_t)fv[1];
    if constexpr (DIM == 3) key_lo[f] = (uint32_t)fv[2];
    face_id[f] = (int32_t)f;
}

__global__ void __launch_bounds__(256) gather_u64_kernel(const uint64_t *__restrict__ src, const int32_t *__restrict__ idx,
                                                          uint64_t *__restrict__ dst, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[idx[i]];
}

// sorted faces: equal neighbours in the sorted order are the two sides of an interior face
template <int DIM>
__global__ void __launch_bounds__(256) pair_faces_kernel(const int32_t *__restrict__ cells, const int32_t *__restrict__ sorted_face,
                                                          int64_t nfaces, int32_t *__restrict__ neigh, int32_t *__restrict__ err)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i + 1 >= nfaces) return;
    int32_t f0 = sorted_face[i], f1 = sorted_face[i + 1];
    int32_t a[DIM], b[DIM];
    face_ids<DIM>(cells, f0 / (DIM + 1), f0 % (DIM + 1), a);
    face_ids<DIM>(cells, f1 / (DIM + 1), f1 % (DIM + 1), b);
    bool same = true;
#pragma unroll
    for (int k = 0; k < DIM; ++k) same = same && (a[k] == b[k]);
    if (!same) return;
    neigh[f0] = f1 / (DIM + 1);
    neigh[f1] = f0 / (DIM + 1);
    if (i + 2 < nfaces) {
        int32_t f2 = sorted_face[i + 2], c[DIM];
        face_ids<DIM>(cells, f2 / (DIM + 1), f2 % (DIM + 1), c);
        bool same2 = true;
#pragma unroll
        for (int k = 0; k < DIM; ++k) same2 = same2 && (a[k] == c[k]);
        if (same2) atomicExch(err, 1);       // a face shared by three cells: not a manifold mesh
    }
}

template <int DIM>
__global__ void __launch_bounds__(256) oppside_kernel(const double *__restrict__ verts, const int32_t *__restrict__ cells,
                                                       int64_t nc, uint8_t *__restrict__ oppside)
{
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nc) return;
    unsigned bits = 0;
#pragma unroll
    for (int j = 0; j <= DIM; ++j) {
        int32_t fv[DIM];
        face_ids<DIM>(cells, c, j, fv);
        double p[DIM];
        const double *v = verts + (int64_t)DIM * cells[c * (DIM + 1) + j];
#pragma unroll
        for (int k = 0; k < DIM; ++k) p[k] = v[k];
        if (face_side<DIM>(verts, fv, p)) bits |= 1u << j;
    }
    oppside[c] = (uint8_t)bits;
}

// per-cell affine map for the integrator's walk: lambda_i = M_i . (p - v0), i = 1..DIM; lambda_0 = 1 - sum
template <int DIM, typename TC> struct alignas(32) CellRec {
    TC M[DIM * DIM];
    TC v0[DIM];
    int32_t vid[DIM + 1];
};

template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cellrec_kernel(const double *__restrict__ verts, const int32_t *__restrict__ cells,
                                                       int64_t nc, CellRec<DIM, TC> *__restrict__ rec)
{
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nc) return;
    const int32_t *cv = cells + c * (DIM + 1);
    const double *v0 = verts + (int64_t)DIM * cv[0];
    CellRec<DIM, TC> r;
    if constexpr (DIM == 2) {
        const double *v1 = verts + 2 * (int64_t)cv[1], *v2 = verts + 2 * (int64_t)cv[2];
        double e1x = v1[0] - v0[0], e1y = v1[1] - v0[1], e2x = v2[0] - v0[0], e2y = v2[1] - v0[1];
        double idet = 1.0 / (e1x * e2y - e1y * e2x);
        r.M[0] = (TC)(e2y * idet);  r.M[1] = (TC)(-e2x * idet);      // lambda_1
        r.M[2] = (TC)(-e1y * idet); r.M[3] = (TC)(e1x * idet);       // lambda_2
    } else {
        const double *v1 = verts + 3 * (int64_t)cv[1], *v2 = verts + 3 * (int64_t)cv[2], *v3 = verts + 3 * (int64_t)cv[3];
        double e1[3], e2[3], e3[3];
        for (int k = 0; k < 3; ++k) { e1[k] = v1[k] - v0[k]; e2[k] = v2[k] - v0[k]; e3[k] = v3[k] - v0[k]; }
        double c23[3] = {e2[1] * e3[2] - e2[2] * e3[1], e2[2] * e3[0] - e2[0] * e3[2], e2[0] * e3[1] - e2[1] * e3[0]};
        double c31[3] = {e3[1] * e1[2] - e3[2] * e1[1], e3[2] * e1[0] - e3[0] * e1[2], e3[0] * e1[1] - e3[1] * e1[0]};
        double c12[3] = {e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0]};
        double idet = 1.0 / (e1[0] * c23[0] + e1[1] * c23[1] + e1[2] * c23[2]);
        for (int k = 0; k < 3; ++k) { r.M[k] = (TC)(c23[k] * idet); r.M[3 + k] = (TC)(c31[k] * idet); r.M[6 + k] = (TC)(c12[k] * idet); }
    }
    for (int k = 0; k < DIM; ++k) r.v0[k] = (TC)v0[k];
    for (int k = 0; k <= DIM; ++k) r.vid[k] = cv[k];
    rec[c] = r;
}

// ---- bin grid: start cell per bin = the cell with the largest id among those whose centroid falls in the
// bin; empty bins are filled by jump flooding with the candidate whose centroid is nearest to the bin centre.
struct BinGrid {
    int nb[3];
    double lo[3], inv[3];
};

template <int DIM> __device__ __forceinline__ void centroid(const double *verts, const int32_t *cells, int64_t c, double *x)
{
#pragma unroll
    for (int k = 0; k < DIM; ++k) x[k] = 0.0;
    for (int i = 0; i <= DIM; ++i) {
        const double *v = verts + (int64_t)DIM * cells[c * (DIM + 1) + i];
#pragma unroll
        for (int k = 0; k < DIM; ++k) x[k] += v[k];
    }
#pragma unroll
    for (int k = 0; k < DIM; ++k) x[k] *= 1.0 / (DIM + 1);
}

template <int DIM> __device__ __forceinline__ int64_t bin_of(const BinGrid &b, const double *x)
{
    int64_t id = 0, mul = 1;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
        double q = floor((x[k] - b.lo[k]) * b.inv[k]);
        int i = q < 0.0 ? 0 : (q > (double)(b.nb[k] - 1) ? b.nb[k] - 1 : (int)q);
        id += mul * i;
        mul *= b.nb[k];
    }
    return id;
}

template <int DIM>
__global__ void __launch_bounds__(256) bin_scatter_kernel(BinGrid b, const double *__restrict__ verts, const int32_t *__restrict__ cells,
                                                           int64_t nc, int32_t *__restrict__ bins)
{
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nc) return;
    double x[DIM];
    centroid<DIM>(verts, cells, c, x);
    atomicMax(bins + bin_of<DIM>(b, x), (int32_t)c);
}

// One jump-flooding pass.  own[id] >= 0: the bin has a cell of its own (never replaced).  Otherwise the bin keeps the
// nearest (centroid to bin centre) of its current candidate and the candidates of the 26 (8) bins at distance `step`.
template <int DIM>
__global__ void __launch_bounds__(256) bin_flood_kernel(BinGrid b, const double *__restrict__ verts, const int32_t *__restrict__ cells,
                                                         const int32_t *__restrict__ own, const int32_t *__restrict__ src,
                                                         int32_t *__restrict__ dst, int step, int64_t nbins)
{
    int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= nbins) return;
    if (own[id] >= 0) { dst[id] = own[id]; return; }
    int ijk[3] = {(int)(id % b.nb[0]), (int)((id / b.nb[0]) % b.nb[1]), (int)(id / ((int64_t)b.nb[0] * b.nb[1]))};
    double ctr[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) ctr[k] = b.lo[k] + (ijk[k] + 0.5) / b.inv[k];
    double best = 1e300;
    int32_t arg = -1;
    const int kz0 = DIM == 3 ? -1 : 0, kz1 = DIM == 3 ? 1 : 0;
    for (int dz = kz0; dz <= kz1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                int x = ijk[0] + dx * step, y = ijk[1] + dy * step, z = ijk[2] + dz * step;
                if (x < 0 || x >= b.nb[0] || y < 0 || y >= b.nb[1] || z < 0 || z >= b.nb[2]) continue;
                int32_t cand = src[x + (int64_t)b.nb[0] * (y + (int64_t)b.nb[1] * z)];
                if (cand < 0) continue;
                double cx[DIM], d2 = 0.0;
                centroid<DIM>(verts, cells, cand, cx);
#pragma unroll
                for (int k = 0; k < DIM; ++k) d2 += (cx[k] - ctr[k]) * (cx[k] - ctr[k]);
                if (d2 < best || (d2 == best && cand > arg)) { best = d2; arg = cand; }
            }
    dst[id] = arg;
}

// ---------------------------------------------------------------------------------------------
// canonical location of one point: bin -> start cell -> walk; hop cap -> brute-force scan (never expected)
template <int DIM>
__device__ __forceinline__ int32_t locate_canonical(const BinGrid &b, const int32_t *__restrict__ bins, const double *__restrict__ verts,
                                                    const int32_t *__restrict__ cells, const int32_t *__restrict__ neigh,
                                                    const uint8_t *__restrict__ oppside, int64_t nc, int64_t hop_cap, const double *p,
                                                    unsigned long long *__restrict__ stats, int64_t start = -1)
{
    // the owner is unique, so any start cell gives the same answer; the bin grid is the default
    int64_t c = start >= 0 ? start : (int64_t)bins[bin_of<DIM>(b, p)];
    if (c < 0) c = 0;
    for (int64_t hop = 0; hop < hop_cap; ++hop) {
        bool beyond;
        int j = walk_probe<DIM>(verts, cells, neigh, oppside, c, p, &beyond);
        int32_t nb = j < 0 ? 0 : (beyond ? -1 : neigh[c * (DIM + 1) + j]);
        if (j < 0 || nb < 0) {
            atomicAdd(stats + 1, (unsigned long long)hop);
            if ((unsigned long long)hop > stats[2]) atomicMax(stats + 2, (unsigned long long)hop);
            return j < 0 ? (int32_t)c : -1;
        }
        c = nb;
    }
    // The deterministic walk hit its cap: it is circling among slivers that are not numerically Delaunay.  A walk that
    // picks a pseudo-random failing face cannot stay in a cycle; the owner it finds is the same unique owner.
    uint32_t rs = (uint32_t)(c * 2654435761u) ^ (uint32_t)__double2loint(p[0]) ^ 0x9e3779b9u;
    for (int64_t hop = 0; hop < 8 * hop_cap; ++hop) {
        const unsigned opp = oppside[c];
        int failing[DIM + 1], nf = 0;
        bool out = false;
#pragma unroll
        for (int j = 0; j <= DIM; ++j) {
            int32_t fv[DIM];
            face_ids<DIM>(cells, c, j, fv);
            bool strict;
            bool sp = face_side<DIM>(verts, fv, p, &strict);
            if (sp != (bool)((opp >> j) & 1u)) {
                failing[nf++] = j;
                if (strict && neigh[c * (DIM + 1) + j] < 0) out = true;
            }
        }
        if (nf == 0 || out) { atomicAdd(stats + 3, 1ull); return nf == 0 ? (int32_t)c : -1; }
        rs = rs * 1664525u + 1013904223u;
        int j = failing[(rs >> 16) % (unsigned)nf];
        int32_t nb = neigh[c * (DIM + 1) + j];
        if (nb < 0) { atomicAdd(stats + 3, 1ull); return -1; }
        c = nb;
    }
    atomicAdd(stats, 1ull);
    for (int64_t k = 0; k < nc; ++k)
        if (first_failing_face<DIM>(verts, cells, oppside, k, p) < 0) return (int32_t)k;
    return -1;
}

template <int DIM>
__global__ void __launch_bounds__(128) simplex_locate_kernel(BinGrid b, const int32_t *__restrict__ bins, const double *__restrict__ verts,
                                                              const int32_t *__restrict__ cells, const int32_t *__restrict__ neigh,
                                                              const uint8_t *__restrict__ oppside, int64_t nc, int64_t hop_cap,
                                                              const double *__restrict__ pos, int64_t n, int32_t *__restrict__ cell,
                                                              double *__restrict__ bary, unsigned long long *__restrict__ stats)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double p[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) p[k] = pos[i * DIM + k];
    int32_t c = locate_canonical<DIM>(b, bins, verts, cells, neigh, oppside, nc, hop_cap, p, stats);
    cell[i] = c;
    if (!bary) return;
    double lam[DIM + 1];
    if (c < 0) {
        for (int k = 0; k <= DIM; ++k) lam[k] = 0.0;
    } else {
        // vertex-0-relative signed-volume ratios (oracle rule O3)
        const int32_t *cv = cells + (int64_t)c * (DIM + 1);
        const double *v0 = verts + (int64_t)DIM * cv[0];
        if constexpr (DIM == 2) {
            const double *v1 = verts + 2 * (int64_t)cv[1], *v2 = verts + 2 * (int64_t)cv[2];
            double e1x = v1[0] - v0[0], e1y = v1[1] - v0[1], e2x = v2[0] - v0[0], e2y = v2[1] - v0[1];
            double px = p[0] - v0[0], py = p[1] - v0[1];
            double tot = e1x * e2y - e1y * e2x;
            lam[1] = (px * e2y - py * e2x) / tot;
            lam[2] = (e1x * py - e1y * px) / tot;
            lam[0] = 1.0 - lam[1] - lam[2];
        } else {
            const double *v1 = verts + 3 * (int64_t)cv[1], *v2 = verts + 3 * (int64_t)cv[2], *v3 = verts + 3 * (int64_t)cv[3];
            double e1[3], e2[3], e3[3], q[3];
            for (int k = 0; k < 3; ++k) { e1[k] = v1[k] - v0[k]; e2[k] = v2[k] - v0[k]; e3[k] = v3[k] - v0[k]; q[k] = p[k] - v0[k]; }
            auto det3 = [](const double *a, const double *bb, const double *cc) {
                return a[0] * (bb[1] * cc[2] - bb[2] * cc[1]) - a[1] * (bb[0] * cc[2] - bb[2] * cc[0]) + a[2] * (bb[0] * cc[1] - bb[1] * cc[0]);
            };
            double tot = det3(e1, e2, e3);
            lam[1] = det3(q, e2, e3) / tot;
            lam[2] = det3(e1, q, e3) / tot;
            lam[3] = det3(e1, e2, q) / tot;
            lam[0] = 1.0 - lam[1] - lam[2] - lam[3];
        }
    }
    for (int k = 0; k <= DIM; ++k) bary[i * (DIM + 1) + k] = lam[k];
}

// ---------------------------------------------------------------------------------------------
// integrator
// tracer record (array of structures, whole 32-byte sectors: one sector for 3D fp32 and 2D fp64).
// meta = completed steps at exit (low 30 bits) | exit flag << 30
template <int DIM, typename TC> struct alignas(16) SimplexTracer {
    TC x[DIM];
    int32_t cell;
    int32_t orig;
    uint32_t meta;
};

template <typename REC> __device__ __forceinline__ REC load_tracer(const REC *p)
{
    REC r;
    constexpr int NQ = sizeof(REC) / 16;
    const int4 *s = reinterpret_cast<const int4 *>(p);
    int4 *d = reinterpret_cast<int4 *>(&r);
#pragma unroll
    for (int k = 0; k < NQ; ++k) d[k] = s[k];
    return r;
}
template <typename REC> __device__ __forceinline__ void store_tracer(REC *p, const REC &r)
{
    constexpr int NQ = sizeof(REC) / 16;
    const int4 *s = reinterpret_cast<const int4 *>(&r);
    int4 *d = reinterpret_cast<int4 *>(p);
#pragma unroll
    for (int k = 0; k < NQ; ++k) d[k] = s[k];
}

// sort key: Morton code of the tracer's bin (bin grid coarsened by `shift`); finished tracers go to the last bin so
// that live tracers stay compacted at the front and whole warps of finished ones retire at once
template <int DIM, typename TC>
__global__ void __launch_bounds__(256) simplex_key_kernel(BinGrid b, const SimplexTracer<DIM, TC> *__restrict__ st, int64_t n, int shift,
                                                           int row_major, uint32_t last_bin, uint32_t *__restrict__ key,
                                                           uint32_t *__restrict__ cnt)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const SimplexTracer<DIM, TC> t = load_tracer(st + i);
    uint32_t k = last_bin;
    if ((t.meta >> 30) == 0) {
        int c[DIM];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            double q = floor(((double)t.x[a] - b.lo[a]) * b.inv[a]);
            int ia = q < 0.0 ? 0 : (q > (double)(b.nb[a] - 1) ? b.nb[a] - 1 : (int)q);
            c[a] = ia >> shift;
        }
        if (row_major) {
            const int m0 = ((b.nb[0] - 1) >> shift) + 1, m1 = ((b.nb[1] - 1) >> shift) + 1;
            k = (uint32_t)c[0] + (uint32_t)m0 * ((uint32_t)c[1] + (DIM == 3 ? (uint32_t)m1 * (uint32_t)c[2] : 0u));
        } else {
            k = bundle::morton<DIM>(c);
        }
        if (k > last_bin - 1) k = last_bin - 1;
    }
    key[i] = k;
    bundle::count_key(cnt, k, last_bin);
}

template <typename TC> struct WalkTol {};
template <> struct WalkTol<float> { static constexpr float eps = 1e-4f; };
template <> struct WalkTol<double> { static constexpr double eps = 1e-10; };

// NBYTES (multiple of 16) from a 32-byte-aligned read-only record into registers: 256-bit loads (sm_100
// ld.global.nc.v8.b32), one L1 request per 32 bytes per lane, plus one 128-bit load for a 16-byte tail.
template <int NBYTES> __device__ __forceinline__ void load_words(const void *src, uint32_t *w)
{
    static_assert(NBYTES % 16 == 0, "records are multiples of 16 bytes");
    const char *p = reinterpret_cast<const char *>(src);
#pragma unroll
    for (int k = 0; k < NBYTES / 32; ++k)
        asm("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
            : "=r"(w[8 * k]), "=r"(w[8 * k + 1]), "=r"(w[8 * k + 2]), "=r"(w[8 * k + 3]), "=r"(w[8 * k + 4]), "=r"(w[8 * k + 5]),
              "=r"(w[8 * k + 6]), "=r"(w[8 * k + 7]) : "l"(p + 32 * k));
    if constexpr (NBYTES % 32 != 0) {
        constexpr int o = NBYTES / 32 * 8;
        asm("ld.global.nc.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w[o]), "=r"(w[o + 1]), "=r"(w[o + 2]), "=r"(w[o + 3]) : "l"(p + 4 * o));
    }
}

template <typename T> __device__ __forceinline__ T word_value(const uint32_t *w, int i)
{
    if constexpr (sizeof(T) == 4) return __uint_as_float(w[i]);
    else return __hiloint2double((int)w[2 * i + 1], (int)w[2 * i]);
}

// The tet/triangle a tracer last evaluated in, kept in registers: its affine map (CellRec) and the two time levels
// {a, b - a} of its vertices.  Consecutive RK4 stage points are a fraction of a cell apart (h |u| ~ 0.4 cells in
// config 4), so most stages find the point still inside the held cell and issue no load at all; a lane that crossed a
// face walks and reloads alone (predicated), which costs L1 wavefronts only for the lines that lane touches.
template <int DIM, typename TV, typename TC> struct HeldSimplex {
    int32_t cell = -1;              // cell whose CellRec is held
    bool vel = false;               // vertex records of `cell` from `pair` are held
    const void *pair = nullptr;
    CellRec<DIM, TC> r;
    TC a[DIM + 1][DIM], d[DIM + 1][DIM];
};

template <int DIM, typename TC> __device__ __forceinline__ void load_cellrec(const CellRec<DIM, TC> *__restrict__ rec, int32_t c,
                                                                            CellRec<DIM, TC> &r)
{
    constexpr int NB = sizeof(CellRec<DIM, TC>);
    uint32_t w[NB / 4];
    load_words<NB>(rec + c, w);
    constexpr int E = sizeof(TC) / 4;
#pragma unroll
    for (int k = 0; k < DIM * DIM; ++k) r.M[k] = word_value<TC>(w, k);
#pragma unroll
    for (int k = 0; k < DIM; ++k) r.v0[k] = word_value<TC>(w, DIM * DIM + k);
#pragma unroll
    for (int k = 0; k <= DIM; ++k) r.vid[k] = (int32_t)w[(DIM * DIM + DIM) * E + k];
}

// both time levels of vertex v: a[0..DIM), d[0..DIM) widened to the compute type
template <int DIM, typename TV, typename TC>
__device__ __forceinline__ void load_vertex(const PairRec<DIM, TV> *__restrict__ rec, int32_t v, TC *a, TC *d)
{
    constexpr int NB = sizeof(PairRec<DIM, TV>);
    constexpr int P = PadOf<DIM>::P;
    uint32_t w[NB / 4];
    load_words<NB>(rec + v, w);
#pragma unroll
    for (int k = 0; k < DIM; ++k) { a[k] = (TC)word_value<TV>(w, k); d[k] = (TC)word_value<TV>(w, P + k); }
}

// Seeds -> tracer records with their canonical cells (flag 2 = outside at t0).  The owner is decided by the canonical fp64
// predicate, as in lcs_locate; to get there cheaply the walk first runs on the per-cell affine maps in the compute type (one
// 64-byte record and a dozen FMAs per hop instead of four fp64 face predicates on gathered vertex coordinates) and hands its
// last cell to the canonical walk; a seed that the affine map places strictly inside its cell, by more than the rounding-error
// bound of its weights, needs no canonical probe at all (the owner is the same: there is no tie to break).
template <int DIM, typename TC>
__global__ void __launch_bounds__(128) simplex_init_kernel(BinGrid b, const int32_t *__restrict__ bins, const double *__restrict__ verts,
                                                            const int32_t *__restrict__ cells, const int32_t *__restrict__ neigh,
                                                            const uint8_t *__restrict__ oppside, const CellRec<DIM, TC> *__restrict__ crec,
                                                            int64_t nc, int64_t hop_cap, const TC *__restrict__ seeds, int64_t n,
                                                            SimplexTracer<DIM, TC> *__restrict__ st, unsigned long long *__restrict__ stats)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    SimplexTracer<DIM, TC> t;
    double p[DIM];
    TC pc[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) { TC v = seeds[i * DIM + k]; t.x[k] = v; pc[k] = v; p[k] = (double)v; }
    int32_t c = bins[bin_of<DIM>(b, p)];
    if (c < 0) c = 0;
    bool certain = false;
    for (int hop = 0; hop < 16; ++hop) {
        CellRec<DIM, TC> r;
        load_cellrec<DIM, TC>(crec, c, r);
        TC q[DIM], sum = TC(0), lmin;
#pragma unroll
        for (int k = 0; k < DIM; ++k) q[k] = pc[k] - r.v0[k];
        int jmin = 0;
        TC lam[DIM + 1];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            TC l = TC(0);
#pragma unroll
            for (int k = 0; k < DIM; ++k) l = fma(r.M[a * DIM + k], q[k], l);
            lam[a + 1] = l;
            sum += l;
        }
        lam[0] = TC(1) - sum;
        lmin = lam[0];
#pragma unroll
        for (int a = 1; a <= DIM; ++a)
            if (lam[a] < lmin) { lmin = lam[a]; jmin = a; }
        if (lmin >= TC(0)) {
            // Certainly the owner?  Rounding-error bound of the weights computed above: the map entries and v0 are roundings of
            // exact values (relative eps each), q and the FMA chain add a few eps of the term magnitudes:
            // |lam_i - exact| <= 8 eps sum_k |M_ik| (|q_k| + |v0_k|) for i >= 1, their sum (+ eps) for lam_0.  A point whose weights
            // all exceed four times their bounds is strictly inside this cell, so the canonical predicate (which has no tie to break
            // there) names the same owner and is skipped; everything nearer to a face goes through it.
            const TC eps = sizeof(TC) == 4 ? TC(5.9604645e-8) : TC(1.1102230246251565e-16);
            TC e0 = eps;
            certain = true;
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                TC e = TC(0);
#pragma unroll
                for (int k = 0; k < DIM; ++k) e = fma(fabs(r.M[a * DIM + k]), fabs(q[k]) + fabs(r.v0[k]), e);
                e *= TC(8) * eps;
                e0 += e;
                certain = certain && lam[a + 1] > TC(4) * e;
            }
            certain = certain && lam[0] > TC(4) * e0;
            break;
        }
        const int32_t nb = __ldg(neigh + (int64_t)c * (DIM + 1) + jmin);
        if (nb < 0) break;
        c = nb;
    }
    if (!certain) c = locate_canonical<DIM>(b, bins, verts, cells, neigh, oppside, nc, hop_cap, p, stats, c);
    t.cell = c;
    t.orig = (int32_t)i;
    t.meta = c < 0 ? (2u << 30) : 0u;
    store_tracer(st + i, t);
}

// What the in-advect walk needs when it gives up: the canonical (fp64) locator of lcs_locate.
struct CanonCtx {
    BinGrid b;
    const int32_t *bins;
    const double *verts;
    const int32_t *cells;
    const int32_t *neigh;
    const uint8_t *oppside;
    int64_t nc, hop_cap;
    unsigned long long *stats;
};

// canonical owner of p (or -1 = outside the mesh)
template <int DIM, typename TC> __device__ __forceinline__ int32_t walk_fallback(const CanonCtx &cx, const TC *p)
{
    double q[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) q[k] = (double)p[k];
    atomicAdd(cx.stats + 5, 1ull);
    return locate_canonical<DIM>(cx.b, cx.bins, cx.verts, cx.cells, cx.neigh, cx.oppside, cx.nc, cx.hop_cap, q, cx.stats + 8);
}

// u(p, tau) with the walk from *cell.  Returns 0 = evaluated, 1 = p left the mesh through a hull face, 2 (SLOW == false
// only) = the walk on the per-cell affine maps (compute type) has not reached a cell that holds p, to the tolerance, within
// kWalkCap hops: a stage point many cells away, or two slivers whose rounded maps each push the point into the other.  The
// integrator then hands the tracer to its SLOW instantiation (a second, small launch over the tracers so marked), which
// locates such a point again with the canonical fp64 predicate of lcs_locate (info key "walk_fallbacks") and interpolates
// in its owner: a tracer is never interpolated in a cell that does not hold it ("walk_cap_hits" stays 0 by construction),
// and the rare path costs the hot kernel neither registers nor code.
constexpr int kWalkCap = 24;
template <int DIM, typename TV, typename TC, bool SLOW, bool ONE_PAIR = false>
__device__ __forceinline__ int simplex_velocity(const CellRec<DIM, TC> *__restrict__ crec, const int32_t *__restrict__ neigh,
                                                 const PairRec<DIM, TV> *__restrict__ vrec, TC tau, const TC *p, int32_t *cell,
                                                 HeldSimplex<DIM, TV, TC> &h, const CanonCtx &cx, TC *u)
{
    int32_t c = *cell;
    TC lam[DIM + 1];
    // ONE_PAIR: every stage of the launch reads the same snapshot pair (the usual window), so the held vertex records can only
    // be stale right after a cell change inside this call: no pair bookkeeping, and the vertex ids die with the reload
    if constexpr (!ONE_PAIR) {
        if (h.pair != (const void *)vrec) { h.vel = false; h.pair = vrec; }    // uniform: another snapshot pair
    }
    bool forced = false, fresh = false;
    for (int hop = 0;; ++hop) {
        if (h.cell != c) {
            load_cellrec<DIM, TC>(crec, c, h.r);
            // the neighbour row of the new cell will be wanted by the next hop out of it: bring its line into L1 now
            asm volatile("prefetch.global.L1 [%0];" ::"l"(neigh + (int64_t)c * (DIM + 1)));
            h.cell = c;
            h.vel = false;
            fresh = true;
        }
        TC q[DIM];
#pragma unroll
        for (int k = 0; k < DIM; ++k) q[k] = p[k] - h.r.v0[k];
        TC sum = TC(0);
#pragma unroll
        for (int i = 0; i < DIM; ++i) {
            TC l = TC(0);
#pragma unroll
            for (int k = 0; k < DIM; ++k) l = fma(h.r.M[i * DIM + k], q[k], l);
            lam[i + 1] = l;
            sum += l;
        }
        lam[0] = TC(1) - sum;
        int jmin = 0;
        TC lmin = lam[0];
#pragma unroll
        for (int i = 1; i <= DIM; ++i)
            if (lam[i] < lmin) { lmin = lam[i]; jmin = i; }
        if (lmin >= -WalkTol<TC>::eps || forced) break;
        if (hop >= kWalkCap) {
            if constexpr (!SLOW) return 2;
            c = walk_fallback<DIM, TC>(cx, p);
            if (c < 0) return 1;
            forced = true;                       // weights of the canonical owner, whatever their rounding
            continue;
        }
        int32_t nb = __ldg(neigh + (int64_t)c * (DIM + 1) + jmin);
        if (nb < 0) return 1;
        c = nb;
    }
    *cell = c;
    if (ONE_PAIR ? fresh : !h.vel) {
#pragma unroll
        for (int i = 0; i <= DIM; ++i) load_vertex<DIM, TV, TC>(vrec, h.r.vid[i], h.a[i], h.d[i]);
        h.vel = true;
    }
#pragma unroll
    for (int k = 0; k < DIM; ++k) u[k] = TC(0);
#pragma unroll
    for (int i = 0; i <= DIM; ++i) {
#pragma unroll
        for (int k = 0; k < DIM; ++k) u[k] = fma(lam[i], fma(tau, h.d[i][k], h.a[i][k]), u[k]);
    }
    return 0;
}

// Tracers whose walk gave up (simplex_velocity returned 2) are parked with flag 3 and their index appended to `pend`; the
// SLOW instantiation, launched right after on the same stream, resumes each of them at the step it stopped in and finishes the
// launch unit with the canonical re-location available.  No other kernel ever sees flag 3.
struct Pending {
    unsigned int *count;      // number of parked tracers of this launch unit (zeroed before the fast launch)
    int32_t *index;           // their slots in the tracer array
};

template <int DIM, typename TV, typename TC, bool SLOW, bool ONE_PAIR = false>
__global__ void __launch_bounds__(128, (SLOW ? 1 : (sizeof(TC) == 4 ? 7 : (DIM == 2 ? 5 : 1))))
simplex_window_kernel(const CellRec<DIM, TC> *__restrict__ crec, const int32_t *__restrict__ neigh, const PairRec<DIM, TV> *__restrict__ pa,
                      const PairRec<DIM, TV> *__restrict__ pb, const PairRec<DIM, TV> *__restrict__ pc, const TC *__restrict__ tau,
                      int nsteps, int first_step, int64_t n, SimplexTracer<DIM, TC> *__restrict__ st, TC h,
                      const __grid_constant__ CanonCtx cx, Pending pend)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = SLOW ? (int64_t)gridDim.x * blockDim.x : n;
    const int64_t count = SLOW ? (int64_t)*pend.count : n;
    if (i >= count) return;
    do {
        const int64_t slot = SLOW ? (int64_t)pend.index[i] : i;
        SimplexTracer<DIM, TC> t = load_tracer(st + slot);
        if ((t.meta >> 30) != (SLOW ? 3u : 0u)) continue;
        TC x[DIM];
#pragma unroll
        for (int k = 0; k < DIM; ++k) x[k] = t.x[k];
        int32_t cell = t.cell;
        int s = SLOW ? (int)(t.meta & 0x3fffffffu) - first_step : 0, rc = 0;
        HeldSimplex<DIM, TV, TC> held;
        for (; s < nsteps; ++s) {
            const TC ta = __ldg(tau + 3 * s), tb = __ldg(tau + 3 * s + 1), tc = __ldg(tau + 3 * s + 2);
            // the running sum k1 + 2 k2 + 2 k3 instead of the four slopes: six registers fewer live at stage 4
            TC acc[DIM], u[DIM], y[DIM];
            int32_t c = cell;
            rc = simplex_velocity<DIM, TV, TC, SLOW, ONE_PAIR>(crec, neigh, pa, ta, x, &c, held, cx, acc);
            if (rc) break;
#pragma unroll
            for (int k = 0; k < DIM; ++k) y[k] = fma(TC(0.5) * h, acc[k], x[k]);
            rc = simplex_velocity<DIM, TV, TC, SLOW, ONE_PAIR>(crec, neigh, pb, tb, y, &c, held, cx, u);
            if (rc) break;
#pragma unroll
            for (int k = 0; k < DIM; ++k) { y[k] = fma(TC(0.5) * h, u[k], x[k]); acc[k] = fma(TC(2), u[k], acc[k]); }
            rc = simplex_velocity<DIM, TV, TC, SLOW, ONE_PAIR>(crec, neigh, pb, tb, y, &c, held, cx, u);
            if (rc) break;
#pragma unroll
            for (int k = 0; k < DIM; ++k) { y[k] = fma(h, u[k], x[k]); acc[k] = fma(TC(2), u[k], acc[k]); }
            rc = simplex_velocity<DIM, TV, TC, SLOW, ONE_PAIR>(crec, neigh, pc, tc, y, &c, held, cx, u);
            if (rc) break;
#pragma unroll
            for (int k = 0; k < DIM; ++k) x[k] = fma(h * TC(1.0 / 6.0), acc[k] + u[k], x[k]);
            cell = c;
        }
#pragma unroll
        for (int k = 0; k < DIM; ++k) t.x[k] = x[k];
        t.cell = cell;
        t.meta = rc ? ((uint32_t)(rc == 2 ? 3u : 1u) << 30) | (uint32_t)(first_step + s) : 0u;
        if (!SLOW && rc == 2) pend.index[atomicAdd(pend.count, 1u)] = (int32_t)slot;
        store_tracer(st + slot, t);
    } while (SLOW && (i += stride) < count);
}

// Adams-Bashforth 4 with an RK4 start-up on simplicial meshes (row f4, reading #31): as simplex_window_kernel,
// one velocity evaluation (walk + interpolation) per step after the first three; hist [n][3][DIM] as in cart_ab4_kernel.
template <int DIM, typename TV, typename TC, bool SLOW>
__global__ void __launch_bounds__(128)
simplex_ab4_kernel(const CellRec<DIM, TC> *__restrict__ crec, const int32_t *__restrict__ neigh, const PairRec<DIM, TV> *__restrict__ pa,
                   const PairRec<DIM, TV> *__restrict__ pb, const PairRec<DIM, TV> *__restrict__ pc, const TC *__restrict__ tau,
                   int nsteps, int first_step, int64_t n, SimplexTracer<DIM, TC> *__restrict__ st, TC *__restrict__ hist, TC h,
                   const __grid_constant__ CanonCtx cx, Pending pend)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = SLOW ? (int64_t)gridDim.x * blockDim.x : n;
    const int64_t count = SLOW ? (int64_t)*pend.count : n;
    if (i >= count) return;
    do {
        const int64_t slot = SLOW ? (int64_t)pend.index[i] : i;
        SimplexTracer<DIM, TC> t = load_tracer(st + slot);
        if ((t.meta >> 30) != (SLOW ? 3u : 0u)) continue;
        int s = SLOW ? (int)(t.meta & 0x3fffffffu) - first_step : 0, rc = 0;
        const bool have_hist = first_step + s > 0;
        TC x[DIM], h0[DIM], h1[DIM], h2[DIM];
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
            x[k] = t.x[k];
            h0[k] = have_hist ? hist[(slot * 3 + 0) * DIM + k] : TC(0);
            h1[k] = have_hist ? hist[(slot * 3 + 1) * DIM + k] : TC(0);
            h2[k] = have_hist ? hist[(slot * 3 + 2) * DIM + k] : TC(0);
        }
        int32_t cell = t.cell;
        HeldSimplex<DIM, TV, TC> held;
        for (; s < nsteps; ++s) {
            const TC ta = __ldg(tau + 3 * s), tb = __ldg(tau + 3 * s + 1), tc = __ldg(tau + 3 * s + 2);
            TC k1[DIM], inc[DIM];
            int32_t c = cell;
            rc = simplex_velocity<DIM, TV, TC, SLOW>(crec, neigh, pa, ta, x, &c, held, cx, k1);
            if (rc) break;
            if (first_step + s < 3) {
                TC k2[DIM], k3[DIM], k4[DIM], y[DIM];
#pragma unroll
                for (int k = 0; k < DIM; ++k) y[k] = fma(TC(0.5) * h, k1[k], x[k]);
                rc = simplex_velocity<DIM, TV, TC, SLOW>(crec, neigh, pb, tb, y, &c, held, cx, k2);
                if (rc) break;
#pragma unroll
                for (int k = 0; k < DIM; ++k) y[k] = fma(TC(0.5) * h, k2[k], x[k]);
                rc = simplex_velocity<DIM, TV, TC, SLOW>(crec, neigh, pb, tb, y, &c, held, cx, k3);
                if (rc) break;
#pragma unroll
                for (int k = 0; k < DIM; ++k) y[k] = fma(h, k3[k], x[k]);
                rc = simplex_velocity<DIM, TV, TC, SLOW>(crec, neigh, pc, tc, y, &c, held, cx, k4);
                if (rc) break;
#pragma unroll
                for (int k = 0; k < DIM; ++k) inc[k] = TC(1.0 / 6.0) * ((k1[k] + k4[k]) + TC(2) * (k2[k] + k3[k]));
            } else {
#pragma unroll
                for (int k = 0; k < DIM; ++k) inc[k] = TC(1.0 / 24.0) * (((TC(55) * k1[k] - TC(59) * h0[k]) + TC(37) * h1[k]) - TC(9) * h2[k]);
            }
#pragma unroll
            for (int k = 0; k < DIM; ++k) {
                x[k] = fma(h, inc[k], x[k]);
                h2[k] = h1[k]; h1[k] = h0[k]; h0[k] = k1[k];
            }
            cell = c;
        }
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
            t.x[k] = x[k];
            hist[(slot * 3 + 0) * DIM + k] = h0[k]; hist[(slot * 3 + 1) * DIM + k] = h1[k]; hist[(slot * 3 + 2) * DIM + k] = h2[k];
        }
        t.cell = cell;
        t.meta = rc ? ((uint32_t)(rc == 2 ? 3u : 1u) << 30) | (uint32_t)(first_step + s) : 0u;
        if (!SLOW && rc == 2) pend.index[atomicAdd(pend.count, 1u)] = (int32_t)slot;
        store_tracer(st + slot, t);
    } while (SLOW && (i += stride) < count);
}

// ---------------------------------------------------------------------------------------------
// Split variant (the paper's design on unstructured grids: "the RK4 computation was divided into several
// short kernels", each velocity evaluation "preceded by a cell search", i.e. 8 kernels per step; integrator option 2).  All
// tracers advance one stage at a time; between the launches the stage point (xi), the running sum k1 + 2 k2 + 2 k3 (acc) and
// the cell found for the stage point (scell) live in global memory as [n] arrays.  A tracer whose stage point leaves the mesh
// gets its flag at once; its record (position and cell at the start of the step) is only rewritten by the last launch of a
// step in which all four evaluations succeeded.  Same arithmetic per evaluation as the fused kernel (walk on the affine maps
// with the canonical re-location when the walk gives up, P1 interpolation, time blend).
template <int DIM, typename TC, int STAGE>
__global__ void __launch_bounds__(128)
simplex_search_kernel(const CellRec<DIM, TC> *__restrict__ crec, const int32_t *__restrict__ neigh, int step, int64_t n,
                      SimplexTracer<DIM, TC> *__restrict__ st, const TC *__restrict__ xi_g, int32_t *__restrict__ scell,
                      const __grid_constant__ CanonCtx cx)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    SimplexTracer<DIM, TC> t = load_tracer(st + i);
    if ((t.meta >> 30) != 0) return;
    TC p[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) p[k] = STAGE == 0 ? t.x[k] : xi_g[i * DIM + k];
    int32_t c = STAGE == 0 ? t.cell : scell[i];
    bool forced = false;
    int rc = 0;
    for (int hop = 0;; ++hop) {
        CellRec<DIM, TC> r;
        load_cellrec<DIM, TC>(crec, c, r);
        TC q[DIM], lam[DIM + 1];
#pragma unroll
        for (int k = 0; k < DIM; ++k) q[k] = p[k] - r.v0[k];
        TC sum = TC(0);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            TC l = TC(0);
#pragma unroll
            for (int k = 0; k < DIM; ++k) l = fma(r.M[a * DIM + k], q[k], l);
            lam[a + 1] = l;
            sum += l;
        }
        lam[0] = TC(1) - sum;
        int jmin = 0;
        TC lmin = lam[0];
#pragma unroll
        for (int a = 1; a <= DIM; ++a)
            if (lam[a] < lmin) { lmin = lam[a]; jmin = a; }
        if (lmin >= -WalkTol<TC>::eps || forced) break;
        if (hop >= kWalkCap) {
            c = walk_fallback<DIM, TC>(cx, p);
            if (c < 0) { rc = 1; break; }
            forced = true;
            continue;
        }
        int32_t nb = __ldg(neigh + (int64_t)c * (DIM + 1) + jmin);
        if (nb < 0) { rc = 1; break; }
        c = nb;
    }
    if (rc) {
        t.meta = (1u << 30) | (uint32_t)step;
        store_tracer(st + i, t);
        return;
    }
    scell[i] = c;
}

template <int DIM, typename TV, typename TC, int STAGE>
__global__ void __launch_bounds__(128)
simplex_interp_kernel(const CellRec<DIM, TC> *__restrict__ crec, const PairRec<DIM, TV> *__restrict__ vrec, TC tau, int64_t n,
                      SimplexTracer<DIM, TC> *__restrict__ st, TC *__restrict__ xi_g, TC *__restrict__ acc_g,
                      const int32_t *__restrict__ scell, TC h)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    SimplexTracer<DIM, TC> t = load_tracer(st + i);
    if ((t.meta >> 30) != 0) return;
    TC p[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) p[k] = STAGE == 0 ? t.x[k] : xi_g[i * DIM + k];
    const int32_t c = scell[i];
    CellRec<DIM, TC> r;
    load_cellrec<DIM, TC>(crec, c, r);
    TC q[DIM], lam[DIM + 1], u[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) q[k] = p[k] - r.v0[k];
    TC sum = TC(0);
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        TC l = TC(0);
#pragma unroll
        for (int k = 0; k < DIM; ++k) l = fma(r.M[a * DIM + k], q[k], l);
        lam[a + 1] = l;
        sum += l;
    }
    lam[0] = TC(1) - sum;
#pragma unroll
    for (int k = 0; k < DIM; ++k) u[k] = TC(0);
#pragma unroll
    for (int a = 0; a <= DIM; ++a) {
        TC va[DIM], vd[DIM];
        load_vertex<DIM, TV, TC>(vrec, r.vid[a], va, vd);
#pragma unroll
        for (int k = 0; k < DIM; ++k) u[k] = fma(lam[a], fma(tau, vd[k], va[k]), u[k]);
    }
    if constexpr (STAGE < 3) {
        const TC cf = STAGE == 2 ? TC(1) : TC(0.5);
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
            xi_g[i * DIM + k] = fma(cf * h, u[k], t.x[k]);
            acc_g[i * DIM + k] = STAGE == 0 ? u[k] : acc_g[i * DIM + k] + TC(2) * u[k];
        }
    } else {
#pragma unroll
        for (int k = 0; k < DIM; ++k) t.x[k] = fma(h * TC(1.0 / 6.0), acc_g[i * DIM + k] + u[k], t.x[k]);
        t.cell = c;                                   // start of the next step's walk
        store_tracer(st + i, t);
    }
}

template <int DIM, typename TC>
__global__ void __launch_bounds__(256) simplex_final_kernel(int64_t n, const SimplexTracer<DIM, TC> *__restrict__ st, int32_t N,
                                                             TC *__restrict__ flowmap, uint8_t *__restrict__ exit_flag,
                                                             int32_t *__restrict__ exit_step)
{
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const SimplexTracer<DIM, TC> t = load_tracer(st + j);
    const int64_t i = t.orig;
    const uint32_t fl = t.meta >> 30;
#pragma unroll
    for (int k = 0; k < DIM; ++k) flowmap[i * DIM + k] = t.x[k];
    if (exit_flag) exit_flag[i] = (uint8_t)fl;
    if (exit_step) exit_step[i] = fl == 0 ? N : (fl == 2 ? 0 : (int32_t)(t.meta & 0x3fffffffu));
}

BinGrid make_bins(const lcs_field *f)
{
    BinGrid b;
    for (int k = 0; k < 3; ++k) { b.nb[k] = f->mesh.nb[k]; b.lo[k] = f->mesh.bin_lo[k]; b.inv[k] = f->mesh.bin_inv[k]; }
    return b;
}

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

template <int DIM> lcs_status build_impl(lcs_field *f, const double *vh, const int32_t *ch)
{
    SimplexMesh &m = f->mesh;
    const int64_t nv = m.nv, nc = m.nc, nf = nc * (DIM + 1);
    // host validation + bounding box
    for (int64_t i = 0; i < nf; ++i)
        if (ch[i] < 0 || ch[i] >= nv) { lcs_set_error("cell %lld has vertex index %d out of range", (long long)(i / (DIM + 1)), ch[i]); return LCS_ERR_MESH; }
    for (int64_t c = 0; c < nc; ++c)
        for (int a = 0; a <= DIM; ++a)
            for (int b2 = a + 1; b2 <= DIM; ++b2)
                if (ch[c * (DIM + 1) + a] == ch[c * (DIM + 1) + b2]) { lcs_set_error("cell %lld repeats a vertex", (long long)c); return LCS_ERR_MESH; }
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t v = 0; v < nv; ++v)
        for (int k = 0; k < DIM; ++k) {
            double x = vh[v * DIM + k];
            if (!isfinite(x)) { lcs_set_error("vertex %lld is not finite", (long long)v); return LCS_ERR_MESH; }
            lo[k] = std::min(lo[k], x); hi[k] = std::max(hi[k], x);
        }
    LCS_CUDA_OK(cudaMalloc((void **)&m.verts, (size_t)nv * DIM * 8));
    LCS_CUDA_OK(cudaMalloc((void **)&m.cells, (size_t)nf * 4));
    LCS_CUDA_OK(cudaMalloc((void **)&m.neigh, (size_t)nf * 4));
    LCS_CUDA_OK(cudaMalloc((void **)&m.oppside, (size_t)nc));
    LCS_CUDA_OK(cudaMalloc((void **)&m.stats, 16 * sizeof(unsigned long long)));
    LCS_CUDA_OK(cudaMemset(m.stats, 0, 16 * sizeof(unsigned long long)));
    LCS_CUDA_OK(cudaMemcpy(m.verts, vh, (size_t)nv * DIM * 8, cudaMemcpyHostToDevice));
    LCS_CUDA_OK(cudaMemcpy(m.cells, ch, (size_t)nf * 4, cudaMemcpyHostToDevice));
    LCS_CUDA_OK(cudaMemset(m.neigh, 0xff, (size_t)nf * 4));
    cudaStream_t st = 0;

    // ---- adjacency: sort face keys (CUB radix sort: set-up, not the hot path), pair equal neighbours
    uint64_t *key_hi = nullptr, *key_hi2 = nullptr;
    uint32_t *key_lo = nullptr, *key_lo2 = nullptr;
    int32_t *fid = nullptr, *fid2 = nullptr, *err = nullptr;
    void *tmp = nullptr;
    auto cleanup = [&]() {
        cudaFree(key_hi); cudaFree(key_hi2); cudaFree(key_lo); cudaFree(key_lo2); cudaFree(fid); cudaFree(fid2); cudaFree(err); cudaFree(tmp);
    };
#define BUILD_OK(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { lcs_set_error("%s: %s", #expr, cudaGetErrorString(e__)); cleanup(); return e__ == cudaErrorMemoryAllocation ? LCS_ERR_OOM : LCS_ERR_CUDA; } } while (0)
    BUILD_OK(cudaMalloc((void **)&key_hi, (size_t)nf * 8));
    BUILD_OK(cudaMalloc((void **)&key_hi2, (size_t)nf * 8));
    BUILD_OK(cudaMalloc((void **)&fid, (size_t)nf * 4));
    BUILD_OK(cudaMalloc((void **)&fid2, (size_t)nf * 4));
    BUILD_OK(cudaMalloc((void **)&err, 4));
    BUILD_OK(cudaMemset(err, 0, 4));
    if (DIM == 3) { BUILD_OK(cudaMalloc((void **)&key_lo, (size_t)nf * 4)); BUILD_OK(cudaMalloc((void **)&key_lo2, (size_t)nf * 4)); }
    LCS_LAUNCH((face_key_kernel<DIM>), lcs_blocks(nf, 256), 256, 0, st, m.cells, nf, key_hi, key_lo, fid);
    size_t tb1 = 0, tb2 = 0;
    if (DIM == 3) cub::DeviceRadixSort::SortPairs(nullptr, tb1, key_lo, key_lo2, fid, fid2, (int)nf, 0, 32, st);
    cub::DeviceRadixSort::SortPairs(nullptr, tb2, key_hi, key_hi2, fid, fid2, (int)nf, 0, 64, st);
    BUILD_OK(cudaMalloc(&tmp, std::max(tb1, tb2)));
    const int32_t *sorted = nullptr;
    if (DIM == 3) {
        // LSD: sort by the third id, then (stable) by the first two
        BUILD_OK(cub::DeviceRadixSort::SortPairs(tmp, tb1, key_lo, key_lo2, fid, fid2, (int)nf, 0, 32, st));
        LCS_LAUNCH(gather_u64_kernel, lcs_blocks(nf, 256), 256, 0, st, key_hi, fid2, key_hi2, nf);
        BUILD_OK(cub::DeviceRadixSort::SortPairs(tmp, tb2, key_hi2, key_hi, fid2, fid, (int)nf, 0, 64, st));
        sorted = fid;
    } else {
        BUILD_OK(cub::DeviceRadixSort::SortPairs(tmp, tb2, key_hi, key_hi2, fid, fid2, (int)nf, 0, 64, st));
        sorted = fid2;
    }
    g_lcs_launches.fetch_add(DIM == 3 ? 2 : 1);
    LCS_LAUNCH((pair_faces_kernel<DIM>), lcs_blocks(nf, 256), 256, 0, st, m.cells, sorted, nf, m.neigh, err);
    int32_t herr = 0;
    BUILD_OK(cudaMemcpy(&herr, err, 4, cudaMemcpyDeviceToHost));
    cleanup();
#undef BUILD_OK
    if (herr) { lcs_set_error("a face is shared by more than two cells"); return LCS_ERR_MESH; }

    LCS_LAUNCH((oppside_kernel<DIM>), lcs_blocks(nc, 256), 256, 0, st, m.verts, m.cells, nc, m.oppside);

    // ---- per-cell affine maps in the compute dtype
    if (f->compute_dtype == LCS_F64) {
        LCS_CUDA_OK(cudaMalloc(&m.cellrec, (size_t)nc * sizeof(CellRec<DIM, double>)));
        LCS_LAUNCH((cellrec_kernel<DIM, double>), lcs_blocks(nc, 256), 256, 0, st, m.verts, m.cells, nc, (CellRec<DIM, double> *)m.cellrec);
    } else {
        LCS_CUDA_OK(cudaMalloc(&m.cellrec, (size_t)nc * sizeof(CellRec<DIM, float>)));
        LCS_LAUNCH((cellrec_kernel<DIM, float>), lcs_blocks(nc, 256), 256, 0, st, m.verts, m.cells, nc, (CellRec<DIM, float> *)m.cellrec);
    }

    // ---- bin grid: about one bin per cell, cubic bins
    double ext[3] = {1, 1, 1}, vol = 1.0;
    for (int k = 0; k < DIM; ++k) { ext[k] = std::max(hi[k] - lo[k], 1e-300); vol *= ext[k]; }
    double target = std::min((double)nc, (double)(1 << 26));
    double hb = pow(vol / target, 1.0 / DIM);
    int64_t nbins = 1;
    for (int k = 0; k < 3; ++k) {
        m.nb[k] = k < DIM ? (int)std::max(1.0, std::min(4096.0, ceil(ext[k] / hb))) : 1;
        m.bin_lo[k] = k < DIM ? lo[k] : 0.0;
        m.bin_inv[k] = k < DIM ? m.nb[k] / ext[k] : 0.0;
        nbins *= m.nb[k];
    }
    int32_t *own = nullptr, *ping = nullptr, *pong = nullptr;
    LCS_CUDA_OK(cudaMalloc((void **)&own, (size_t)nbins * 4));
    LCS_CUDA_OK(cudaMalloc((void **)&ping, (size_t)nbins * 4));
    LCS_CUDA_OK(cudaMalloc((void **)&pong, (size_t)nbins * 4));
    LCS_CUDA_OK(cudaMemset(own, 0xff, (size_t)nbins * 4));
    BinGrid b = make_bins(f);
    LCS_LAUNCH((bin_scatter_kernel<DIM>), lcs_blocks(nc, 256), 256, 0, st, b, m.verts, m.cells, nc, own);
    LCS_CUDA_OK(cudaMemcpyAsync(ping, own, (size_t)nbins * 4, cudaMemcpyDeviceToDevice, st));
    int maxnb = std::max(m.nb[0], std::max(m.nb[1], m.nb[2]));
    int step = 1;
    while (step * 2 < maxnb) step *= 2;
    for (; step >= 1; step /= 2) {                 // jump flooding, then two more unit passes
        LCS_LAUNCH((bin_flood_kernel<DIM>), lcs_blocks(nbins, 256), 256, 0, st, b, m.verts, m.cells, own, ping, pong, step, nbins);
        std::swap(ping, pong);
    }
    for (int extra = 0; extra < 2; ++extra) {
        LCS_LAUNCH((bin_flood_kernel<DIM>), lcs_blocks(nbins, 256), 256, 0, st, b, m.verts, m.cells, own, ping, pong, 1, nbins);
        std::swap(ping, pong);
    }
    LCS_CUDA_OK(cudaDeviceSynchronize());
    m.bins = ping;
    cudaFree(pong);
    cudaFree(own);
    m.hop_cap = (int64_t)(4.0 * pow((double)nc, 1.0 / DIM)) + 64;
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

// how lcs_advect carves the scratch on a simplicial mesh (shared with lcs_field_reserve, see CartLayout)
struct SimplexLayout {
    bool ab4, split, do_bundle;
    int shift;
    int64_t nbins, ntiles;
    size_t o_a, o_b, o_tau, o_hist, o_xi, o_acc, o_scell, o_key, o_cnt, o_tile, o_pend, total;
};

size_t simplex_tracer_bytes(const lcs_field *f)
{
    const bool c64 = f->compute_dtype == LCS_F64;
    if (f->dim == 2) return c64 ? sizeof(SimplexTracer<2, double>) : sizeof(SimplexTracer<2, float>);
    return c64 ? sizeof(SimplexTracer<3, double>) : sizeof(SimplexTracer<3, float>);
}

SimplexLayout simplex_layout(const lcs_field *f, int64_t n, int64_t N)
{
    SimplexLayout L{};
    const SimplexMesh &m = f->mesh;
    const int DIM = f->dim;
    const size_t tcb = lcs_esize(f->compute_dtype), trb = simplex_tracer_bytes(f);
    // re-bundling by bin (Morton or row-major order of the coarsened bin grid), histogram <= 2^24 bins
    L.ab4 = f->opt_integrator == 3;
    L.split = f->opt_integrator == 2;
    L.do_bundle = !L.ab4 && (f->opt_bundle == 1 || (f->opt_bundle < 0 && n >= (1 << 18)));
    int bits = 0;
    for (L.shift = 0;; ++L.shift) {
        bits = 0;
        for (int a = 0; a < DIM; ++a) {
            int cells = ((m.nb[a] - 1) >> L.shift) + 1, b = 0;
            while ((1 << b) < cells) ++b;
            bits = b > bits ? b : bits;
        }
        if (bits * DIM <= 24) break;
    }
    L.nbins = L.do_bundle ? ((int64_t)1 << (bits * DIM)) + 1 : 0;
    L.ntiles = (L.nbins + bundle::kScanTile - 1) / bundle::kScanTile;
    size_t off = 0;
    L.o_a = off; off = align_up(off + (size_t)n * trb);
    L.o_b = off; if (L.do_bundle) off = align_up(off + (size_t)n * trb);
    L.o_tau = off; off = align_up(off + (size_t)3 * N * tcb);
    L.o_hist = off; if (L.ab4) off = align_up(off + (size_t)n * 3 * DIM * tcb);
    L.o_xi = off; if (L.split) off = align_up(off + (size_t)n * DIM * tcb);
    L.o_acc = off; if (L.split) off = align_up(off + (size_t)n * DIM * tcb);
    L.o_scell = off; if (L.split) off = align_up(off + (size_t)n * 4);
    L.o_key = off; if (L.do_bundle) off = align_up(off + (size_t)n * 4);
    L.o_cnt = off; if (L.do_bundle) off = align_up(off + (size_t)L.nbins * 4);
    L.o_tile = off; if (L.do_bundle) off = align_up(off + (size_t)L.ntiles * 4);
    L.o_pend = off; off = align_up(off + 256 + (size_t)n * 4);      // counter + slots of the tracers handed to the slow path
    L.total = off;
    return L;
}

template <int DIM, typename TV, typename TC>
lcs_status simplex_advect_impl(lcs_field *f, int64_t n, const void *seeds_, double t0, double h, int64_t N, void *flowmap_,
                               uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st)
{
    using Tracer = SimplexTracer<DIM, TC>;
    const TC *seeds = (const TC *)seeds_;
    TC *flowmap = (TC *)flowmap_;
    SimplexMesh &m = f->mesh;
    if (n >= (1LL << 31) || N >= (1LL << 24)) { lcs_set_error("too many seeds or steps for 32-bit tracer records"); return LCS_ERR_INVALID_ARG; }
    std::vector<StepWindow> windows;
    lcs_status rc = lcs_plan_windows(f, t0, h, N, windows);
    if (rc != LCS_OK) return rc;
    const SimplexLayout L = simplex_layout(f, n, N);
    rc = lcs_scratch_check(f, L.total);
    if (rc != LCS_OK) return rc;
    const bool ab4 = L.ab4, do_bundle = L.do_bundle;
    const int64_t nbins = L.nbins;
    char *base = (char *)f->scratch.buf;
    Tracer *cur = (Tracer *)(base + L.o_a), *alt = (Tracer *)(base + L.o_b);
    TC *d_tau = (TC *)(base + L.o_tau);
    uint32_t *d_key = (uint32_t *)(base + L.o_key), *d_cnt = (uint32_t *)(base + L.o_cnt), *d_tile = (uint32_t *)(base + L.o_tile);
    BinGrid b = make_bins(f);
    const CanonCtx cx{b, m.bins, m.verts, m.cells, m.neigh, m.oppside, m.nc, m.hop_cap, m.stats};
    LCS_LAUNCH((simplex_init_kernel<DIM, TC>), lcs_blocks(n, 128), 128, 0, st, b, m.bins, m.verts, m.cells, m.neigh, m.oppside,
               (const CellRec<DIM, TC> *)m.cellrec, m.nc, m.hop_cap, seeds, n, cur, m.stats);
    const int block = f->opt_block ? (int)(f->opt_block > 128 ? 128 : f->opt_block) : 128;
    const int dir = h > 0 ? 1 : -1;
    using VRec = PairRec<DIM, TV>;
    int64_t since_bundle = -1;                       // -1: not bundled yet
    // unstructured meshes: tracers cross a cell in ~2.5 steps but stay spatially coherent much longer, and a sort moves
    // every record: re-bundle every 160 steps unless told otherwise (measured on config 4: 160 > per window > once)
    const int64_t bundle_every = f->opt_bundle_steps > 0 ? f->opt_bundle_steps : 160;
    for (size_t wi = 0; wi < windows.size(); ++wi) {
        const StepWindow &w = windows[wi];
        const void *p[3];
        for (int k = 0; k < 3; ++k) {
            rc = lcs_field_require_pair(f, w.s[k], st, &p[k]);
            if (rc != LCS_OK) return rc;
        }
        // stage-time weights of the window's steps, computed on the device (no host-to-device copy in the hot call)
        rc = lcs_fill_stage_tau(f, t0, h, w.first, w.count, w.s, d_tau, nullptr, st);
        if (rc != LCS_OK) return rc;
        lcs_field_prefetch(f, dir > 0 ? w.s[2] + 2 : w.s[2] - 1, w.s[2], w.s[2] + 1);
        const int chunk = (do_bundle && f->opt_bundle_steps > 0 && f->opt_bundle_steps < w.count) ? (int)f->opt_bundle_steps : w.count;
        for (int done = 0, cnt = 0; done < w.count; done += cnt) {
            cnt = lcs_early_cut(f, w.first + done, w.count - done < chunk ? w.count - done : chunk);
            const int first = (int)w.first + done;
            if (do_bundle && (since_bundle < 0 || since_bundle >= bundle_every)) {
                LCS_CUDA_OK(cudaMemsetAsync(d_cnt, 0, (size_t)nbins * 4, st));
                LCS_LAUNCH((simplex_key_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, b, cur, n, L.shift, (int)f->opt_simplex_order, (uint32_t)(nbins - 1), d_key, d_cnt);
                bundle::sort_records<Tracer>(cur, alt, d_key, d_cnt, d_tile, n, nbins, st);
                std::swap(cur, alt);
                since_bundle = 0;
            }
            since_bundle += cnt;
            if (L.split) {
                // the paper's 8 launches per RK4 step: search + interpolate for each of the four evaluations
                WindowTimer timer(f, st);
                TC *xi = (TC *)(base + L.o_xi), *acc = (TC *)(base + L.o_acc);
                int32_t *scell = (int32_t *)(base + L.o_scell);
                const CellRec<DIM, TC> *cr = (const CellRec<DIM, TC> *)m.cellrec;
                const unsigned grid = lcs_blocks(n, block);
                for (int sstep = first; sstep < first + cnt; ++sstep) {
                    const TC t3[3] = {(TC)lcs_stage_tau(f, t0, h, sstep, 0, w.s[0]), (TC)lcs_stage_tau(f, t0, h, sstep, 1, w.s[1]),
                                      (TC)lcs_stage_tau(f, t0, h, sstep, 2, w.s[2])};
                    LCS_LAUNCH((simplex_search_kernel<DIM, TC, 0>), grid, block, 0, st, cr, m.neigh, sstep, n, cur, xi, scell, cx);
                    LCS_LAUNCH((simplex_interp_kernel<DIM, TV, TC, 0>), grid, block, 0, st, cr, (const VRec *)p[0], t3[0], n, cur, xi, acc, scell, (TC)h);
                    LCS_LAUNCH((simplex_search_kernel<DIM, TC, 1>), grid, block, 0, st, cr, m.neigh, sstep, n, cur, xi, scell, cx);
                    LCS_LAUNCH((simplex_interp_kernel<DIM, TV, TC, 1>), grid, block, 0, st, cr, (const VRec *)p[1], t3[1], n, cur, xi, acc, scell, (TC)h);
                    LCS_LAUNCH((simplex_search_kernel<DIM, TC, 2>), grid, block, 0, st, cr, m.neigh, sstep, n, cur, xi, scell, cx);
                    LCS_LAUNCH((simplex_interp_kernel<DIM, TV, TC, 2>), grid, block, 0, st, cr, (const VRec *)p[1], t3[1], n, cur, xi, acc, scell, (TC)h);
                    LCS_LAUNCH((simplex_search_kernel<DIM, TC, 3>), grid, block, 0, st, cr, m.neigh, sstep, n, cur, xi, scell, cx);
                    LCS_LAUNCH((simplex_interp_kernel<DIM, TV, TC, 3>), grid, block, 0, st, cr, (const VRec *)p[2], t3[2], n, cur, xi, acc, scell, (TC)h);
                }
            } else {
            const Pending pend{(unsigned int *)(base + L.o_pend), (int32_t *)(base + L.o_pend + 256)};
            LCS_CUDA_OK(cudaMemsetAsync(pend.count, 0, 4, st));
            {
                WindowTimer timer(f, st);
                if (ab4)
                    LCS_LAUNCH((simplex_ab4_kernel<DIM, TV, TC, false>), lcs_blocks(n, block), block, 0, st, (const CellRec<DIM, TC> *)m.cellrec, m.neigh,
                               (const VRec *)p[0], (const VRec *)p[1], (const VRec *)p[2], d_tau + 3 * (size_t)first, cnt, first, n, cur,
                               (TC *)(base + L.o_hist), (TC)h, cx, pend);
                else if (p[0] == p[1] && p[1] == p[2])
                    LCS_LAUNCH((simplex_window_kernel<DIM, TV, TC, false, true>), lcs_blocks(n, block), block, 0, st, (const CellRec<DIM, TC> *)m.cellrec, m.neigh,
                               (const VRec *)p[0], (const VRec *)p[1], (const VRec *)p[2], d_tau + 3 * (size_t)first, cnt, first, n, cur, (TC)h, cx, pend);
                else
                    LCS_LAUNCH((simplex_window_kernel<DIM, TV, TC, false>), lcs_blocks(n, block), block, 0, st, (const CellRec<DIM, TC> *)m.cellrec, m.neigh,
                               (const VRec *)p[0], (const VRec *)p[1], (const VRec *)p[2], d_tau + 3 * (size_t)first, cnt, first, n, cur, (TC)h, cx, pend);
            }
            // the tracers whose walk gave up (usually none): a small grid-stride launch over the parked slots
            if (ab4)
                LCS_LAUNCH((simplex_ab4_kernel<DIM, TV, TC, true>), 148, 128, 0, st, (const CellRec<DIM, TC> *)m.cellrec, m.neigh,
                           (const VRec *)p[0], (const VRec *)p[1], (const VRec *)p[2], d_tau + 3 * (size_t)first, cnt, first, n, cur,
                           (TC *)(base + L.o_hist), (TC)h, cx, pend);
            else
                LCS_LAUNCH((simplex_window_kernel<DIM, TV, TC, true>), 148, 128, 0, st, (const CellRec<DIM, TC> *)m.cellrec, m.neigh,
                           (const VRec *)p[0], (const VRec *)p[1], (const VRec *)p[2], d_tau + 3 * (size_t)first, cnt, first, n, cur, (TC)h, cx, pend);
            }
            if (lcs_early_due(f, (int64_t)first + cnt, N)) {         // row f1: evaluate C for the stencils that are still complete
                LCS_LAUNCH((simplex_final_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, n, cur, (int32_t)N, (TC *)f->early.flowmap,
                           f->early.flag, (int32_t *)nullptr);
                rc = lcs_early_cg_eval(f, (int64_t)first + cnt, st);
                if (rc != LCS_OK) return rc;
            }
        }
        f->info_windows++;
    }
    LCS_LAUNCH((simplex_final_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, n, cur, (int32_t)N, flowmap, exit_flag, exit_step);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

}  // namespace

size_t lcs_simplex_scratch_bytes(const lcs_field *f, int64_t n, int64_t N) { return simplex_layout(f, n, N).total; }

lcs_status lcs_simplex_build(lcs_field *f, const double *verts_host, const int32_t *cells_host)
{
    return f->dim == 2 ? build_impl<2>(f, verts_host, cells_host) : build_impl<3>(f, verts_host, cells_host);
}

void lcs_simplex_free(lcs_field *f)
{
    SimplexMesh &m = f->mesh;
    if (m.verts) cudaFree(m.verts);
    if (m.cells) cudaFree(m.cells);
    if (m.neigh) cudaFree(m.neigh);
    if (m.oppside) cudaFree(m.oppside);
    if (m.cellrec) cudaFree(m.cellrec);
    if (m.bins) cudaFree(m.bins);
    if (m.stats) cudaFree(m.stats);
    m = SimplexMesh();
}

lcs_status lcs_simplex_locate(lcs_field *f, int64_t n, const double *pos, int32_t *cell, double *bary, cudaStream_t st)
{
    SimplexMesh &m = f->mesh;
    BinGrid b = make_bins(f);
    if (f->dim == 2)
        LCS_LAUNCH((simplex_locate_kernel<2>), lcs_blocks(n, 128), 128, 0, st, b, m.bins, m.verts, m.cells, m.neigh, m.oppside, m.nc, m.hop_cap, pos, n, cell, bary, m.stats);
    else
        LCS_LAUNCH((simplex_locate_kernel<3>), lcs_blocks(n, 128), 128, 0, st, b, m.bins, m.verts, m.cells, m.neigh, m.oppside, m.nc, m.hop_cap, pos, n, cell, bary, m.stats);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

lcs_status lcs_simplex_advect(lcs_field *f, int64_t n, const void *seeds, double t0, double h, int64_t N, void *flowmap,
                              uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st)
{
    const bool v64 = f->vel_dtype == LCS_F64, c64 = f->compute_dtype == LCS_F64;
    if (f->dim == 2) {
        if (v64 && c64) return simplex_advect_impl<2, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && c64) return simplex_advect_impl<2, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && !c64) return simplex_advect_impl<2, float, float>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    } else {
        if (v64 && c64) return simplex_advect_impl<3, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && c64) return simplex_advect_impl<3, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && !c64) return simplex_advect_impl<3, float, float>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    }
    lcs_set_error("fp64 velocity with fp32 arithmetic is not supported (compute_dtype must be >= vel_dtype)");
    return LCS_ERR_INVALID_ARG;
}
