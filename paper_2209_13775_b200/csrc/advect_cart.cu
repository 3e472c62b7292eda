// advect_cart.cu -- Cartesian grids: cell search by arithmetic indexing (row a1), bi/trilinear space +
// linear time interpolation (row a3) and the RK4 integrator (row a4), for sm_100a.
//
// Paper: RK4 needs "the vector field to be evaluated at 4 different locations in space-time for a single
// update step"; both space and time interpolation run on the GPU between the two frames of
// the current window; the run time is in the interpolation gathers and is bandwidth-bound
// (PAPER.md:77, 91).
//
// Design (differs from the paper's Kepler kernels):
//  * a tracer is (cell index, fractional offset in [0,1)) per axis, in grid units.  The offset is what the
//    interpolation weights need, the index is what the gather addresses need, periodic wrap is a mask on
//    the index and never touches the stored position, and an fp32 offset carries ~1e-7 of a CELL instead
//    of ~1e-7 of the domain.  Physical positions exist only at the API boundary (fp64 conversion).
//  * the tracer state is one 32-byte record (array of structures): one sector in, one sector out per
//    launch, and re-bundling moves whole sectors.
//  * gathers read "pair records" {a, b-a}: both time levels of a node in one 32-byte sector (one 256-bit
//    load), the time blend is one FMA per component.  The record array is padded by one node per axis so
//    that the 2^d corners of a cell sit at constant offsets from one base address.
//  * tracers are re-bundled by cell once per snapshot window, in row-major cell order (x fastest; Morton order is the
//    other option): the kernel is bound by L1 wavefronts, a load costs one wavefront per distinct 128-byte line that
//    each group of 4 lanes touches, and x-neighbouring cells share a line (profiles/r1_cfg3_baseline.md).
//  * 3D fp32: the time blend is hoisted out of the gather into per-stage-time "x-pair" fields and the corners of the
//    last gathered cell stay in registers (cart_xpair_kernel below).
//  * fused variant: one thread runs every RK4 step of a snapshot window; split variant (the paper's): one
//    short kernel per RK4 stage with the stage state in global memory.
#include <limits.h>
#include <math.h>

#include <algorithm>

#include "bundle_sort.cuh"
#include "lcs_internal.cuh"

namespace {

struct CartDev {
    int n[3];
    int periodic[3];
    int pow2[3];
    int np0, np01;         // padded record strides (CartGeom::np): np0 = np[0], np01 = np[0] * np[1]
    double origin[3], spacing[3], inv[3];
};

// tracer record.  meta = completed steps at exit (low 30 bits) | exit flag << 30
template <int DIM, typename TC> struct alignas(16) CartTracer {
    TC w[DIM];
    int32_t ci[DIM];
    int32_t orig;
    uint32_t meta;
};
static_assert(sizeof(CartTracer<3, float>) == 32 && sizeof(CartTracer<2, double>) == 32, "one sector per tracer");

template <typename REC> __device__ __forceinline__ REC load_record(const REC *p)
{
    REC r;
    constexpr int NQ = sizeof(REC) / 16;
    const int4 *s = reinterpret_cast<const int4 *>(p);
    int4 *d = reinterpret_cast<int4 *>(&r);
#pragma unroll
    for (int k = 0; k < NQ; ++k) d[k] = s[k];
    return r;
}
template <typename REC> __device__ __forceinline__ void store_record(REC *p, const REC &r)
{
    constexpr int NQ = sizeof(REC) / 16;
    const int4 *s = reinterpret_cast<const int4 *>(&r);
    int4 *d = reinterpret_cast<int4 *>(p);
#pragma unroll
    for (int k = 0; k < NQ; ++k) d[k] = s[k];
}

// time-blended velocity at one node: out = a + tau * d  (one FMA per component).  LD256: the 32-byte record is
// fetched with one 256-bit load (sm_100 ld.global.v8.b32 / v4.b64), i.e. one L1 request per corner.
template <int DIM, typename TV, typename TC, bool LD256>
__device__ __forceinline__ void node_velocity(const PairRec<DIM, TV> *__restrict__ p, TC tau, TC *out)
{
    if constexpr (DIM == 3 && sizeof(TV) == 4) {
        float4 a, d;
        if constexpr (LD256) {
            asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(d.x), "=f"(d.y), "=f"(d.z), "=f"(d.w) : "l"(p));
        } else {
            const float4 *q = reinterpret_cast<const float4 *>(p);
            a = __ldg(q); d = __ldg(q + 1);
        }
        out[0] = fma(tau, (TC)d.x, (TC)a.x);
        out[1] = fma(tau, (TC)d.y, (TC)a.y);
        out[2] = fma(tau, (TC)d.z, (TC)a.z);
    } else if constexpr (DIM == 3) {
        double2 a0, a1, d0, d1;
        if constexpr (LD256) {
            asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a0.x), "=d"(a0.y), "=d"(a1.x), "=d"(a1.y) : "l"(p));
            asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(d0.x), "=d"(d0.y), "=d"(d1.x), "=d"(d1.y)
                : "l"(reinterpret_cast<const char *>(p) + 32));
        } else {
            const double2 *q = reinterpret_cast<const double2 *>(p);
            a0 = __ldg(q); a1 = __ldg(q + 1); d0 = __ldg(q + 2); d1 = __ldg(q + 3);
        }
        out[0] = fma(tau, (TC)d0.x, (TC)a0.x);
        out[1] = fma(tau, (TC)d0.y, (TC)a0.y);
        out[2] = fma(tau, (TC)d1.x, (TC)a1.x);
    } else if constexpr (sizeof(TV) == 8) {
        double2 a, d;
        if constexpr (LD256) {
            asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a.x), "=d"(a.y), "=d"(d.x), "=d"(d.y) : "l"(p));
        } else {
            const double2 *q = reinterpret_cast<const double2 *>(p);
            a = __ldg(q); d = __ldg(q + 1);
        }
        out[0] = fma(tau, (TC)d.x, (TC)a.x);
        out[1] = fma(tau, (TC)d.y, (TC)a.y);
    } else {
        float4 r = __ldg(reinterpret_cast<const float4 *>(p));
        out[0] = fma(tau, (TC)r.z, (TC)r.x);
        out[1] = fma(tau, (TC)r.w, (TC)r.y);
    }
}

__device__ __forceinline__ int wrap_index(int c, int n, int pow2)
{
    if (pow2) return c & (n - 1);
    int r = c % n;
    return r < 0 ? r + n : r;
}

// x -> (floor(x) as int, x - floor(x)).  fp32: floor through an add rounded toward -inf onto 1.5 * 2^23, whose low mantissa
// bits then hold the integer (exact for |x| < 2^22 cells): three FP32-pipe instructions instead of FRND + F2I on the
// quarter-rate conversion unit.
template <typename TC> __device__ __forceinline__ void floor_split(TC x, int &ifl, TC &frac)
{
    if constexpr (sizeof(TC) == 4) {
        const float t = __fadd_rd(x, 12582912.0f);
        ifl = __float_as_int(t) - 0x4B400000;
        frac = x - (t - 12582912.0f);
    } else {
        const TC f = floor(x);
        ifl = (int)f;
        frac = x - f;
    }
}

// u(x,t) at the point (ci + xi) in grid units, xi = offset relative to the tracer's cell (any magnitude).
// Returns false if the point is outside a non-periodic axis (closed upper end, as in oracle rule O2).
// FASTWRAP: every axis periodic with a power-of-two node count (mask wrap, no branches).
template <int DIM, typename TV, typename TC, bool FASTWRAP, bool LD256>
__device__ __forceinline__ bool cart_velocity(const CartDev &g, const PairRec<DIM, TV> *__restrict__ rec, TC tau,
                                              const int *ci, const TC *xi, TC *u)
{
    int lo[DIM];
    TC wl[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int ifl;
        floor_split<TC>(xi[a], ifl, wl[a]);
        int c = ci[a] + ifl;
        if constexpr (FASTWRAP) {
            lo[a] = c & (g.n[a] - 1);
        } else if (g.periodic[a]) {
            lo[a] = wrap_index(c, g.n[a], g.pow2[a]);
        } else {
            if (c == g.n[a] - 1 && wl[a] == TC(0)) { c = g.n[a] - 2; wl[a] = TC(1); }
            if (c < 0 || c > g.n[a] - 2) return false;
            lo[a] = c;
        }
    }
    using Rec = PairRec<DIM, TV>;
    if constexpr (DIM == 2) {
        const Rec *b = rec + (lo[0] + lo[1] * g.np0);
        TC v00[2], v10[2], v01[2], v11[2];
        node_velocity<2, TV, TC, LD256>(b, tau, v00);
        node_velocity<2, TV, TC, LD256>(b + 1, tau, v10);
        node_velocity<2, TV, TC, LD256>(b + g.np0, tau, v01);
        node_velocity<2, TV, TC, LD256>(b + g.np0 + 1, tau, v11);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            TC a0 = fma(wl[0], v10[c] - v00[c], v00[c]);
            TC a1 = fma(wl[0], v11[c] - v01[c], v01[c]);
            u[c] = fma(wl[1], a1 - a0, a0);
        }
    } else {
        const Rec *b = rec + (lo[0] + lo[1] * g.np0 + lo[2] * g.np01);
        TC v[8][3];
        node_velocity<3, TV, TC, LD256>(b, tau, v[0]);
        node_velocity<3, TV, TC, LD256>(b + 1, tau, v[1]);
        node_velocity<3, TV, TC, LD256>(b + g.np0, tau, v[2]);
        node_velocity<3, TV, TC, LD256>(b + g.np0 + 1, tau, v[3]);
        node_velocity<3, TV, TC, LD256>(b + g.np01, tau, v[4]);
        node_velocity<3, TV, TC, LD256>(b + g.np01 + 1, tau, v[5]);
        node_velocity<3, TV, TC, LD256>(b + g.np01 + g.np0, tau, v[6]);
        node_velocity<3, TV, TC, LD256>(b + g.np01 + g.np0 + 1, tau, v[7]);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            TC a00 = fma(wl[0], v[1][c] - v[0][c], v[0][c]);
            TC a10 = fma(wl[0], v[3][c] - v[2][c], v[2][c]);
            TC a01 = fma(wl[0], v[5][c] - v[4][c], v[4][c]);
            TC a11 = fma(wl[0], v[7][c] - v[6][c], v[6][c]);
            TC b0 = fma(wl[1], a10 - a00, a00);
            TC b1 = fma(wl[1], a11 - a01, a01);
            u[c] = fma(wl[2], b1 - b0, b0);
        }
    }
    return true;
}

// ---------------------------------------------------------------------------------------------
// seeds (physical, compute dtype) -> (cell, offset) state.  fp64 arithmetic, the oracle's O2 formula, so
// the initial cell agrees with lcs_locate.  flag 2 = seed outside at t0.
// sort key of a live tracer (the orders are described at cart_key_kernel below)
template <int DIM, typename TC>
__device__ __forceinline__ uint32_t cart_key_of(const CartDev &g, const int *ci, const TC *w, int shift, int order, uint32_t last_bin)
{
    int c[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) c[a] = (g.periodic[a] ? wrap_index(ci[a], g.n[a], g.pow2[a]) : ci[a]) >> shift;
    const int m0 = ((g.n[0] - 1) >> shift) + 1, m1 = ((g.n[1] - 1) >> shift) + 1;
    uint32_t k;
    if (order == 2 && DIM == 3) {
        const uint32_t m0p = (uint32_t)(m0 + 1) >> 1;
        const uint32_t sub = ((w[DIM - 1] >= TC(0.5)) ? 8u : 0u) | ((w[1] >= TC(0.5)) ? 4u : 0u) | (((uint32_t)c[0] & 1u) << 1) |
                             ((w[0] >= TC(0.5)) ? 1u : 0u);
        k = (((uint32_t)c[0] >> 1) + m0p * ((uint32_t)c[1] + (uint32_t)m1 * (uint32_t)c[DIM - 1])) * 16u + sub;
    } else if (order == 3 && DIM == 3) {
        // bricks of 4 x 2 x 2 cells, x fastest inside and across bricks: 256 consecutive tracers then sit in a box of about
        // 8 x 2 x 2 cells, whose records the staged integrator copies into shared memory as one small tile
        const uint32_t mb0 = (uint32_t)(m0 + 3) >> 2, mb1 = (uint32_t)(m1 + 1) >> 1;
        const uint32_t sub = ((uint32_t)c[0] & 3u) | (((uint32_t)c[1] & 1u) << 2) | (((uint32_t)c[DIM - 1] & 1u) << 3);
        k = (((uint32_t)c[0] >> 2) + mb0 * (((uint32_t)c[1] >> 1) + mb1 * ((uint32_t)c[DIM - 1] >> 1))) * 16u + sub;
    } else if (order >= 1) {
        k = (uint32_t)c[0] + (uint32_t)m0 * ((uint32_t)c[1] + (DIM == 3 ? (uint32_t)m1 * (uint32_t)c[DIM - 1] : 0u));
    } else {
        k = bundle::morton<DIM>(c);
    }
    return k > last_bin - 1 ? last_bin - 1 : k;
}

struct KeyOut {                 // where a kernel leaves the sort key of its record for the NEXT re-bundling (key == nullptr: nowhere)
    uint32_t *key, *cnt;
    int shift, order;
    uint32_t last_bin;
};

template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cart_init_kernel(CartDev g, const TC *__restrict__ seeds, int64_t n,
                                                         CartTracer<DIM, TC> *__restrict__ st, int32_t orig_base = 0, KeyOut ko = KeyOut{})
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    CartTracer<DIM, TC> t;
    uint32_t fl = 0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double xi = ((double)seeds[i * DIM + a] - g.origin[a]) * g.inv[a];
        double f = floor(xi);
        int c = (int)f;
        double w = xi - f;
        if (!g.periodic[a]) {
            if (!(xi >= 0.0 && xi <= (double)(g.n[a] - 1))) { fl = 2; c = 0; w = 0; }
            else if (c == g.n[a] - 1) { c = g.n[a] - 2; w = 1.0; }
        }
        t.ci[a] = c;
        t.w[a] = (TC)w;
    }
    t.orig = orig_base + (int32_t)i;
    t.meta = fl << 30;
    store_record(st + i, t);
    if (ko.key) {
        const uint32_t k = fl ? ko.last_bin : cart_key_of<DIM, TC>(g, t.ci, t.w, ko.shift, ko.order, ko.last_bin);
        ko.key[i] = k;
        bundle::count_key(ko.cnt, k, ko.last_bin);
    }
}

// (cell, offset) -> physical flow map + flags, scattered back to the caller's seed order
template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cart_final_kernel(CartDev g, const TC *__restrict__ seeds, int64_t n,
                                                          const CartTracer<DIM, TC> *__restrict__ st, int32_t N,
                                                          TC *__restrict__ flowmap, uint8_t *__restrict__ exit_flag,
                                                          int32_t *__restrict__ exit_step)
{
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const CartTracer<DIM, TC> t = load_record(st + j);
    const int64_t i = t.orig;
    const uint32_t fl = t.meta >> 30;
    TC out[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        if (fl == 2) out[a] = seeds[i * DIM + a];
        else out[a] = (TC)(g.origin[a] + ((double)t.ci[a] + (double)t.w[a]) * g.spacing[a]);
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) flowmap[i * DIM + a] = out[a];
    if (exit_flag) exit_flag[i] = (uint8_t)fl;
    if (exit_step) exit_step[i] = fl == 0 ? N : (fl == 2 ? 0 : (int32_t)(t.meta & 0x3fffffffu));
}

// sort key of a tracer; finished tracers (flag != 0) go to the last bin so that their warps retire at once.
// order 0: Morton code of the (wrapped) cell, coarsened by `shift` bits per axis; order 1: row-major cell index, x fastest
// (x-neighbouring cells share a 128-byte line of records).  order 2 (3D, shift == 0): row-major over PAIRS of x-neighbouring
// cells, and inside a pair by (z half, y half, x quarter) of the tracer's offset: a 256-bit gather costs one L1 wavefront per
// distinct 128-byte line that each group of 4 lanes touches, and with 8 tracers per cell in arbitrary order every group
// straddles two rows in y about half of the time (13 instead of 8 wavefronts per request, profiles/r1_cfg3_final.md);
// ordered like this the 4 lanes of a group are x-neighbours in one (y, z) row.
template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cart_key_kernel(CartDev g, const CartTracer<DIM, TC> *__restrict__ st, int64_t n, int shift,
                                                        int order, uint32_t last_bin, uint32_t *__restrict__ key,
                                                        uint32_t *__restrict__ cnt)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const CartTracer<DIM, TC> t = load_record(st + i);
    uint32_t k = last_bin;
    if ((t.meta >> 30) == 3u) { key[i] = bundle::kDropKey; return; }       // record of a finished series volume: dropped by the sort
    if ((t.meta >> 30) == 0) k = cart_key_of<DIM, TC>(g, t.ci, t.w, shift, order, last_bin);
    key[i] = k;
    bundle::count_key(cnt, k, last_bin);
}

// ---------------------------------------------------------------------------------------------
// Fused variant: one thread = one tracer, every RK4 step of the window.  hs[a] = h / spacing[a] turns a
// physical velocity into cells per step.  tau: [nsteps][3] time weights of (ta, tb, tc).
template <int DIM, typename TV, typename TC, bool FASTWRAP, bool LD256>
__global__ void __launch_bounds__(256)
cart_window_kernel(const __grid_constant__ CartDev g, const PairRec<DIM, TV> *__restrict__ pa,
                   const PairRec<DIM, TV> *__restrict__ pb, const PairRec<DIM, TV> *__restrict__ pc,
                   const TC *__restrict__ tau, int nsteps, int first_step, int64_t n, CartTracer<DIM, TC> *__restrict__ st,
                   TC hs0, TC hs1, TC hs2)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    CartTracer<DIM, TC> t = load_record(st + i);
    if ((t.meta >> 30) != 0) return;
    const TC hs[3] = {hs0, hs1, hs2};
    int ci[DIM];
    TC w[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) { ci[a] = t.ci[a]; w[a] = t.w[a]; }
    int s = 0;
    bool ok = true;
    for (; s < nsteps; ++s) {
        const TC ta = __ldg(tau + 3 * s), tb = __ldg(tau + 3 * s + 1), tc = __ldg(tau + 3 * s + 2);
        TC k1[DIM], k2[DIM], k3[DIM], k4[DIM], xi[DIM];
        ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pa, ta, ci, w, k1);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) xi[a] = fma(TC(0.5) * hs[a], k1[a], w[a]);
        ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pb, tb, ci, xi, k2);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) xi[a] = fma(TC(0.5) * hs[a], k2[a], w[a]);
        ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pb, tb, ci, xi, k3);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) xi[a] = fma(hs[a], k3[a], w[a]);
        ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pc, tc, ci, xi, k4);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            TC wn = fma(hs[a] * TC(1.0 / 6.0), (k1[a] + k4[a]) + TC(2) * (k2[a] + k3[a]), w[a]);
            int ifl;
            floor_split<TC>(wn, ifl, w[a]);
            ci[a] += ifl;
        }
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) { t.ci[a] = ci[a]; t.w[a] = w[a]; }
    if (!ok) t.meta = (1u << 30) | (uint32_t)(first_step + s);
    store_record(st + i, t);
}

// ---------------------------------------------------------------------------------------------
// Pre-blended variant (3D, fp32): the time blend u(node, t) = a + tau (b - a) does not depend on the tracer, and the
// integrator is bound by the bytes the L1 delivers into registers (128 B per cycle per SM), so the blend is hoisted
// out of the gather: for a chunk of k RK4 steps the 2k+1 distinct stage times are blended once per node into
// "x-pair" records {u(i0,i1,i2), u(i0+1,i1,i2) - u(i0,i1,i2)} (2 x float4 = one 32-byte sector, one 256-bit load), and a stage
// gathers 4 records = 128 B per tracer instead of 8 pair records = 256 B.  The arithmetic per tracer is unchanged
// (fma(tau, b - a, a) per node, then the nested lerps), so results are bit-identical to the pair-record path.
struct alignas(32) XPair {
    float lo[4];           // u(i0, i1, i2) at the field's stage time
    float hi[4];           // u(i0+1, i1, i2) - u(i0, i1, i2): the x-lerp is one FMA
};

constexpr int kMaxBlendFields = 2 * 256 + 1;

// one thread per padded record; raw snapshots a, b are [node][3] fp32; field f of the chunk gets tau[f]
__global__ void __launch_bounds__(256) blend_xpair_kernel(const float *__restrict__ a, const float *__restrict__ b, int n0, int n1, int n2,
                                                           int q0, int q1, int q2,
                                                           const float *__restrict__ tau, int nfields, XPair *__restrict__ fields,
                                                           int64_t field_stride)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t p0 = q0, p1 = q1, p2 = q2;
    if (i >= p0 * p1 * p2) return;
    int i0 = (int)(i % p0) % n0, i1 = (int)((i / p0) % p1) % n1, i2 = (int)(i / (p0 * p1)) % n2;
    const int j0 = i0 + 1 == n0 ? 0 : i0 + 1;
    const int64_t row = (int64_t)n0 * (i1 + (int64_t)n1 * i2);
    const float *al = a + 3 * (row + i0), *bl = b + 3 * (row + i0), *ah = a + 3 * (row + j0), *bh = b + 3 * (row + j0);
    float va[6], vd[6];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        va[c] = al[c]; vd[c] = bl[c] - al[c];
        va[3 + c] = ah[c]; vd[3 + c] = bh[c] - ah[c];
    }
    for (int f = 0; f < nfields; ++f) {
        const float t = __ldg(tau + f);
        float4 lo, hi;
        lo.x = fmaf(t, vd[0], va[0]); lo.y = fmaf(t, vd[1], va[1]); lo.z = fmaf(t, vd[2], va[2]); lo.w = 0.f;
        hi.x = fmaf(t, vd[3], va[3]) - lo.x; hi.y = fmaf(t, vd[4], va[4]) - lo.y; hi.z = fmaf(t, vd[5], va[5]) - lo.z; hi.w = 0.f;
        // one 256-bit streaming store: a whole 32-byte sector per lane
        asm volatile("st.global.cs.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(fields + (int64_t)f * field_stride + i), "f"(lo.x),
                     "f"(lo.y), "f"(lo.z), "f"(lo.w), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w)
                     : "memory");
    }
}

// L1::no_allocate: a blended field is read by a tracer neighbourhood for two stages and never again, so its lines only evict what
// the SM could reuse; served from L2 without allocation the gathers are 3% (8 tracers per cell) to 7% (30 per cell) faster
__device__ __forceinline__ void load_xpair(const XPair *p, float4 &lo, float4 &hi)
{
    asm("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(lo.x), "=f"(lo.y), "=f"(lo.z), "=f"(lo.w), "=f"(hi.x), "=f"(hi.y), "=f"(hi.z), "=f"(hi.w) : "l"(p));
}

// Corner values of the cell a tracer last gathered from, kept in registers: stages 2 and 3 of a step read the same
// blended field, and so do stage 4 and stage 1 of the next step, at points that are O(h^2) apart -- almost always the
// same cell.  A lane reloads (predicated, per lane) only when its cell changed, which halves the L1 traffic per step.
struct HeldCell {
    int idx;               // record index of the held cell, -1 = nothing held
    float v[8][3];
};

template <bool FASTWRAP, bool REUSE>
__device__ __forceinline__ bool cart_velocity_xpair(const CartDev &g, const XPair *__restrict__ field, const int *ci, const float *xi,
                                                    HeldCell &hc, float *u)
{
    int lo[3];
    float wl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int ifl;
        floor_split<float>(xi[a], ifl, wl[a]);
        int c = ci[a] + ifl;
        if constexpr (FASTWRAP) {
            lo[a] = c & (g.n[a] - 1);
        } else if (g.periodic[a]) {
            lo[a] = wrap_index(c, g.n[a], g.pow2[a]);
        } else {
            if (c == g.n[a] - 1 && wl[a] == 0.f) { c = g.n[a] - 2; wl[a] = 1.f; }
            if (c < 0 || c > g.n[a] - 2) return false;
            lo[a] = c;
        }
    }
    const int idx = lo[0] + lo[1] * g.np0 + lo[2] * g.np01;
    if (!REUSE || idx != hc.idx) {
        const XPair *b = field + idx;
        float4 l00, h00, l10, h10, l01, h01, l11, h11;
        load_xpair(b, l00, h00);
        load_xpair(b + g.np0, l10, h10);
        load_xpair(b + g.np01, l01, h01);
        load_xpair(b + g.np01 + g.np0, l11, h11);
        hc.v[0][0] = l00.x; hc.v[0][1] = l00.y; hc.v[0][2] = l00.z;
        hc.v[1][0] = h00.x; hc.v[1][1] = h00.y; hc.v[1][2] = h00.z;
        hc.v[2][0] = l10.x; hc.v[2][1] = l10.y; hc.v[2][2] = l10.z;
        hc.v[3][0] = h10.x; hc.v[3][1] = h10.y; hc.v[3][2] = h10.z;
        hc.v[4][0] = l01.x; hc.v[4][1] = l01.y; hc.v[4][2] = l01.z;
        hc.v[5][0] = h01.x; hc.v[5][1] = h01.y; hc.v[5][2] = h01.z;
        hc.v[6][0] = l11.x; hc.v[6][1] = l11.y; hc.v[6][2] = l11.z;
        hc.v[7][0] = h11.x; hc.v[7][1] = h11.y; hc.v[7][2] = h11.z;
        hc.idx = idx;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        float a00 = fmaf(wl[0], hc.v[1][c], hc.v[0][c]);       // v[odd] holds the x-difference rounded in fp32 by the blend kernel
        float a10 = fmaf(wl[0], hc.v[3][c], hc.v[2][c]);
        float a01 = fmaf(wl[0], hc.v[5][c], hc.v[4][c]);
        float a11 = fmaf(wl[0], hc.v[7][c], hc.v[6][c]);
        float b0 = fmaf(wl[1], a10 - a00, a00);
        float b1 = fmaf(wl[1], a11 - a01, a01);
        u[c] = fmaf(wl[2], b1 - b0, b0);
    }
    return true;
}

// What the integrator does for a time series (lcs_advect_series) beyond integrating: records carry their own step count, every
// record leaves its sort key for the next re-bundling (no separate key kernel over the set), and the records of the volume that
// finishes with this launch (orig in [fin_lo, fin_hi)) write their outputs and drop out (no separate scan of the set).
struct SeriesTail {
    KeyOut ko;
    int32_t fin_lo, fin_hi, N;
    const float *seeds;
    float *flowmap;
    uint8_t *exit_flag;
    int32_t *exit_step;
};

__device__ __forceinline__ void series_finish(const CartDev &g, const SeriesTail &sr, const CartTracer<3, float> &t)
{
    const uint32_t fl = t.meta >> 30;
    const int64_t i = t.orig;
#pragma unroll
    for (int a = 0; a < 3; ++a)
        sr.flowmap[i * 3 + a] = fl == 2 ? sr.seeds[(i - sr.fin_lo) * 3 + a] : (float)(g.origin[a] + ((double)t.ci[a] + (double)t.w[a]) * g.spacing[a]);
    if (sr.exit_flag) sr.exit_flag[i] = (uint8_t)fl;
    if (sr.exit_step) sr.exit_step[i] = fl == 0 ? sr.N : (fl == 2 ? 0 : (int32_t)(t.meta & 0x3fffffffu));
}

// Step s of the chunk reads the blended fields 2s (ta), 2s+1 (tb), 2s+2 (tc = ta of step s+1): the host only uses this
// kernel for chunks whose stage times have exactly that structure, so the field addresses are warp-uniform arithmetic.
template <bool FASTWRAP, bool SERIES>
__global__ void __launch_bounds__(256)
cart_xpair_kernel(const __grid_constant__ CartDev g, const XPair *__restrict__ fields, int64_t field_stride,
                  int nsteps, int first_step, int64_t n, CartTracer<3, float> *__restrict__ st, float hs0, float hs1, float hs2,
                  const __grid_constant__ SeriesTail sr)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    CartTracer<3, float> t = load_record(st + i);
    if ((t.meta >> 30) != 0) {
        if constexpr (SERIES) {                                // a parked record of the set: it still needs its key, or its exit
            if (sr.ko.key) {
                const bool fin = t.orig >= sr.fin_lo && t.orig < sr.fin_hi;
                if (fin) series_finish(g, sr, t);
                const uint32_t k = fin ? bundle::kDropKey : sr.ko.last_bin;
                sr.ko.key[i] = k;
                if (!fin) bundle::count_key(sr.ko.cnt, k, sr.ko.last_bin);
            }
        }
        return;
    }
    // series mode: tracers of several volumes, each at its own step count, share the launch: a live record carries the steps it
    // has completed in the low bits of meta (otherwise those are zero while the tracer lives)
    if constexpr (SERIES) first_step = (int)(t.meta & 0x3fffffffu);
    const float hs[3] = {hs0, hs1, hs2};
    int ci[3];
    float w[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { ci[a] = t.ci[a]; w[a] = t.w[a]; }
    int s = 0;
    bool ok = true;
    HeldCell hc;
    hc.idx = -1;
    const XPair *held_field = nullptr;
    for (; s < nsteps; ++s) {
        const XPair *fa = fields + (int64_t)(2 * s) * field_stride;
        const XPair *fb = fa + field_stride;
        const XPair *fc = fb + field_stride;
        float k1[3], k2[3], k3[3], k4[3], xi[3];
        if (fa != held_field) hc.idx = -1;                     // uniform: tc of the previous step is ta of this one
        ok = cart_velocity_xpair<FASTWRAP, true>(g, fa, ci, w, hc, k1);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < 3; ++a) xi[a] = fmaf(0.5f * hs[a], k1[a], w[a]);
        ok = cart_velocity_xpair<FASTWRAP, false>(g, fb, ci, xi, hc, k2);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < 3; ++a) xi[a] = fmaf(0.5f * hs[a], k2[a], w[a]);
        ok = cart_velocity_xpair<FASTWRAP, true>(g, fb, ci, xi, hc, k3);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < 3; ++a) xi[a] = fmaf(hs[a], k3[a], w[a]);
        ok = cart_velocity_xpair<FASTWRAP, false>(g, fc, ci, xi, hc, k4);
        held_field = fc;
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float wn = fmaf(hs[a] * (1.0f / 6.0f), (k1[a] + k4[a]) + 2.0f * (k2[a] + k3[a]), w[a]);
            int ifl;
            floor_split<float>(wn, ifl, w[a]);
            ci[a] += ifl;
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) { t.ci[a] = ci[a]; t.w[a] = w[a]; }
    if (!ok) t.meta = (1u << 30) | (uint32_t)(first_step + s);
    else if (SERIES) t.meta = (uint32_t)(first_step + nsteps);
    if constexpr (SERIES) {
        if (sr.ko.key) {
            const bool fin = t.orig >= sr.fin_lo && t.orig < sr.fin_hi;
            if (fin) {
                series_finish(g, sr, t);
                sr.ko.key[i] = bundle::kDropKey;
                return;                                        // the record is not needed any more
            }
            const uint32_t k = ok ? cart_key_of<3, float>(g, ci, w, sr.ko.shift, sr.ko.order, sr.ko.last_bin) : sr.ko.last_bin;
            sr.ko.key[i] = k;
            bundle::count_key(sr.ko.cnt, k, sr.ko.last_bin);
        }
    }
    store_record(st + i, t);
}

// series mode: outputs of the records of one finished volume (orig in [lo, hi)), written to the volume-major output arrays at index
// orig; the records are then marked dead (flag 3) and dropped by the next re-bundling
template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cart_final_series_kernel(CartDev g, const TC *__restrict__ seeds, int64_t n_act, CartTracer<DIM, TC> *__restrict__ st,
                                                                 int32_t lo, int32_t hi, int32_t N, TC *__restrict__ flowmap,
                                                                 uint8_t *__restrict__ exit_flag, int32_t *__restrict__ exit_step)
{
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_act) return;
    CartTracer<DIM, TC> t = load_record(st + j);
    const uint32_t fl = t.meta >> 30;
    if (fl == 3u || t.orig < lo || t.orig >= hi) return;
    const int64_t i = t.orig;
    TC out[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        if (fl == 2) out[a] = seeds[(i - lo) * DIM + a];
        else out[a] = (TC)(g.origin[a] + ((double)t.ci[a] + (double)t.w[a]) * g.spacing[a]);
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) flowmap[i * DIM + a] = out[a];
    if (exit_flag) exit_flag[i] = (uint8_t)fl;
    if (exit_step) exit_step[i] = fl == 0 ? N : (fl == 2 ? 0 : (int32_t)(t.meta & 0x3fffffffu));
    t.meta = 3u << 30;
    store_record(st + j, t);
}

// ---------------------------------------------------------------------------------------------
// Staged variant of the pre-blended integrator (BASELINE.json north_star, second subsystem: "the two bracketing snapshots
// staged through L2 and shared memory via TMA or cp.async"; PAPER.md:61 the window of frames on the GPU, PAPER.md:109 bundles
// "to improve memory coherence and shared-memory GPU performance").  A block owns 256 consecutive tracers of the brick-ordered
// bundle (sort order 3), i.e. a box of about 8 x 2 x 2 cells.  Every RK4 step the block reduces the bounding box of its tracers'
// cells (redux.sync + shared-memory atomics, one barrier), and warp 0 copies the records of that box, grown by the one cell a
// stage point can move, of the two NEW stage-time fields of the step (tb, tc) into shared memory with the TMA engine's
// non-tensor bulk copies (cp.async.bulk.shared.global, one per x-row segment, completion on an mbarrier per field).  Stages 2
// and 4 then gather their 2 x 2 x-pair records from shared memory (8 LDS.128 per lane) instead of the L1; stage 1 and 3 reuse
// the held cell as in cart_xpair_kernel and reload the few lanes that changed cell.  A box larger than the tile capacity
// (a block that straddles the end of a brick row, or tracers that dispersed) and a stage point outside the box fall back to
// the global-memory gather of cart_xpair_kernel, so the result is bit-identical to it in every case.
// Only for grids that are periodic with power-of-two node counts on every axis (no exits; wrap by mask).
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LCS_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LCS_DONE_%=;\n"
        "bra LCS_WAIT_%=;\n"
        "LCS_DONE_%=:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// global -> shared bulk copy by the TMA engine (SASS UBLKCP), bytes a multiple of 16, completion counted on the mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void lds_xpair(uint32_t addr, float4 &lo, float4 &hi)
{
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(lo.x), "=f"(lo.y), "=f"(lo.z), "=f"(lo.w) : "r"(addr));
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(hi.x), "=f"(hi.y), "=f"(hi.z), "=f"(hi.w) : "r"(addr + 16u));
}

struct StageTile {
    uint32_t addr;         // shared-memory address of the tile, 0 = this step is not staged
    int o[3];              // cell coordinates (in the block's local frame) of record 0
    int e[3];              // records per axis
};

__device__ __forceinline__ void set_held(HeldCell &hc, const float4 &l00, const float4 &h00, const float4 &l10, const float4 &h10, const float4 &l01,
                                         const float4 &h01, const float4 &l11, const float4 &h11)
{
    hc.v[0][0] = l00.x; hc.v[0][1] = l00.y; hc.v[0][2] = l00.z;
    hc.v[1][0] = h00.x; hc.v[1][1] = h00.y; hc.v[1][2] = h00.z;
    hc.v[2][0] = l10.x; hc.v[2][1] = l10.y; hc.v[2][2] = l10.z;
    hc.v[3][0] = h10.x; hc.v[3][1] = h10.y; hc.v[3][2] = h10.z;
    hc.v[4][0] = l01.x; hc.v[4][1] = l01.y; hc.v[4][2] = l01.z;
    hc.v[5][0] = h01.x; hc.v[5][1] = h01.y; hc.v[5][2] = h01.z;
    hc.v[6][0] = l11.x; hc.v[6][1] = l11.y; hc.v[6][2] = l11.z;
    hc.v[7][0] = h11.x; hc.v[7][1] = h11.y; hc.v[7][2] = h11.z;
}

// as cart_velocity_xpair<true, REUSE> with the gather served from the shared-memory tile when the cell lies inside it.
// ci = cell in the block's local frame (wrapped once at load, then free-running), hc.idx = packed wrapped cell.
template <bool REUSE>
__device__ __forceinline__ void cart_velocity_staged(const CartDev &g, const XPair *__restrict__ field, const StageTile &tl, const int *ci,
                                                     const float *xi, HeldCell &hc, float *u)
{
    int c[3];
    float wl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int ifl;
        floor_split<float>(xi[a], ifl, wl[a]);
        c[a] = ci[a] + ifl;
    }
    const int key = (c[0] & 1023) | ((c[1] & 1023) << 10) | ((c[2] & 1023) << 20);
    if (!REUSE || key != hc.idx) {
        const int j0 = c[0] - tl.o[0], j1 = c[1] - tl.o[1], j2 = c[2] - tl.o[2];
        float4 l00, h00, l10, h10, l01, h01, l11, h11;
        if (tl.addr != 0u && (unsigned)j0 < (unsigned)tl.e[0] && (unsigned)j1 < (unsigned)(tl.e[1] - 1) && (unsigned)j2 < (unsigned)(tl.e[2] - 1)) {
            const uint32_t sy = (uint32_t)tl.e[0] * 32u, sz = sy * (uint32_t)tl.e[1];
            const uint32_t b = tl.addr + (uint32_t)j0 * 32u + (uint32_t)j1 * sy + (uint32_t)j2 * sz;
            lds_xpair(b, l00, h00);
            lds_xpair(b + sy, l10, h10);
            lds_xpair(b + sz, l01, h01);
            lds_xpair(b + sz + sy, l11, h11);
        } else {
            const XPair *b = field + ((c[0] & (g.n[0] - 1)) + (c[1] & (g.n[1] - 1)) * g.np0 + (c[2] & (g.n[2] - 1)) * g.np01);
            load_xpair(b, l00, h00);
            load_xpair(b + g.np0, l10, h10);
            load_xpair(b + g.np01, l01, h01);
            load_xpair(b + g.np01 + g.np0, l11, h11);
        }
        set_held(hc, l00, h00, l10, h10, l01, h01, l11, h11);
        hc.idx = key;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        float a00 = fmaf(wl[0], hc.v[1][k], hc.v[0][k]);
        float a10 = fmaf(wl[0], hc.v[3][k], hc.v[2][k]);
        float a01 = fmaf(wl[0], hc.v[5][k], hc.v[4][k]);
        float a11 = fmaf(wl[0], hc.v[7][k], hc.v[6][k]);
        float b0 = fmaf(wl[1], a10 - a00, a00);
        float b1 = fmaf(wl[1], a11 - a01, a01);
        u[k] = fmaf(wl[2], b1 - b0, b0);
    }
}

constexpr int kStageBlock = 256;

__global__ void __launch_bounds__(kStageBlock, 4)
cart_xpair_tma_kernel(const __grid_constant__ CartDev g, const XPair *__restrict__ fields, int64_t field_stride, int nsteps, int first_step,
                      int64_t n, CartTracer<3, float> *__restrict__ st, float hs0, float hs1, float hs2, int cap)
{
    extern __shared__ __align__(128) unsigned char smem[];
    // layout: tile of tb | tile of tc | 2 mbarriers | 3 bounding boxes {min[3], max[3], pad[2]}
    const uint32_t tile_b = smem_u32(smem), tile_c = tile_b + (uint32_t)cap * 32u;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + (size_t)cap * 64);
    int *sbox = reinterpret_cast<int *>(smem + (size_t)cap * 64 + 16);
    const uint32_t bar_b = smem_u32(bars), bar_c = bar_b + 8u;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        mbar_init(bar_b, 32);
        mbar_init(bar_c, 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
        for (int k = 0; k < 3; ++k) { sbox[k] = INT_MAX; sbox[3 + k] = INT_MIN; }
    }
    __syncthreads();

    const int64_t i = (int64_t)blockIdx.x * blockDim.x + tid;
    CartTracer<3, float> t;
    bool live = i < n;
    if (live) { t = load_record(st + i); live = (t.meta >> 30) == 0; }
    const float hs[3] = {hs0, hs1, hs2};
    int ci[3] = {0, 0, 0};
    float w[3] = {0.f, 0.f, 0.f};
    if (live) {
#pragma unroll
        for (int a = 0; a < 3; ++a) { ci[a] = t.ci[a] & (g.n[a] - 1); w[a] = t.w[a]; }
    }
    HeldCell hc;
    hc.idx = -1;
    uint32_t uses = 0;                                          // staged steps so far: mbarrier phase parity
    for (int s = 0; s < nsteps; ++s) {
        const XPair *fa = fields + (int64_t)(2 * s) * field_stride;
        const XPair *fb = fa + field_stride;
        const XPair *fc = fb + field_stride;
        // ---- bounding box of the block's cells at the start of the step
        int *box = sbox + 8 * (s % 3);
        {
            const int lo0 = __reduce_min_sync(0xffffffffu, live ? ci[0] : INT_MAX), hi0 = __reduce_max_sync(0xffffffffu, live ? ci[0] : INT_MIN);
            const int lo1 = __reduce_min_sync(0xffffffffu, live ? ci[1] : INT_MAX), hi1 = __reduce_max_sync(0xffffffffu, live ? ci[1] : INT_MIN);
            const int lo2 = __reduce_min_sync(0xffffffffu, live ? ci[2] : INT_MAX), hi2 = __reduce_max_sync(0xffffffffu, live ? ci[2] : INT_MIN);
            if (lane == 0) {
                atomicMin(box + 0, lo0); atomicMin(box + 1, lo1); atomicMin(box + 2, lo2);
                atomicMax(box + 3, hi0); atomicMax(box + 4, hi1); atomicMax(box + 5, hi2);
            }
            if (tid == 0) {
                int *nxt = sbox + 8 * ((s + 1) % 3);
#pragma unroll
                for (int k = 0; k < 3; ++k) { nxt[k] = INT_MAX; nxt[3 + k] = INT_MIN; }
            }
        }
        __syncthreads();                                        // box complete; every thread is done with the tiles of step s - 1
        StageTile tb, tc;
        {
            const int lo0 = box[0], lo1 = box[1], lo2 = box[2], hi0 = box[3], hi1 = box[4], hi2 = box[5];
            // a stage point is less than one cell from the start of the step (checked per lane): x needs cells lo-1 .. hi+1 (the
            // x+1 node is inside the record), y and z need rows lo-1 .. hi+2
            tb.o[0] = lo0 - 1; tb.o[1] = lo1 - 1; tb.o[2] = lo2 - 1;
            tb.e[0] = hi0 - lo0 + 3; tb.e[1] = hi1 - lo1 + 4; tb.e[2] = hi2 - lo2 + 4;
            const bool staged = hi0 >= lo0 && (int64_t)tb.e[0] * tb.e[1] * tb.e[2] <= (int64_t)cap && tb.e[0] <= g.n[0];
            tb.addr = staged ? tile_b : 0u;
            tc = tb;
            tc.addr = staged ? tile_c : 0u;
        }
        const bool staged = tb.addr != 0u;
        if (staged && warp == 0) {
            // one bulk copy per x-row segment and field; a row that crosses the periodic seam in x takes two
            const int rows = tb.e[1] * tb.e[2];
            const int gx = tb.o[0] & (g.n[0] - 1);
            const int n_a = min(tb.e[0], g.n[0] - gx), n_b = tb.e[0] - n_a;
            int mine = 0;
            for (int r = lane; r < rows; r += 32) ++mine;
            const uint32_t bytes = (uint32_t)mine * (uint32_t)tb.e[0] * 32u;
            mbar_arrive_expect_tx(bar_b, bytes);
            mbar_arrive_expect_tx(bar_c, bytes);
            for (int r = lane; r < rows; r += 32) {
                const int jz = r / tb.e[1], jy = r - jz * tb.e[1];
                const int64_t row = (int64_t)((tb.o[1] + jy) & (g.n[1] - 1)) * g.np0 + (int64_t)((tb.o[2] + jz) & (g.n[2] - 1)) * g.np01;
                const uint32_t d = (uint32_t)r * (uint32_t)tb.e[0] * 32u;
                bulk_g2s(tile_b + d, fb + row + gx, (uint32_t)n_a * 32u, bar_b);
                if (n_b > 0) bulk_g2s(tile_b + d + (uint32_t)n_a * 32u, fb + row, (uint32_t)n_b * 32u, bar_b);
                bulk_g2s(tile_c + d, fc + row + gx, (uint32_t)n_a * 32u, bar_c);
                if (n_b > 0) bulk_g2s(tile_c + d + (uint32_t)n_a * 32u, fc + row, (uint32_t)n_b * 32u, bar_c);
            }
        }
        const uint32_t parity = uses & 1u;
        if (staged) ++uses;
        StageTile none;
        none.addr = 0u;
        float k1[3], k2[3], k3[3], k4[3], xi[3];
        // stage 1 reads the field stage 4 of the previous step read: held cell, else (first step, changed cell) global memory
        if (live) {
            cart_velocity_staged<true>(g, fa, none, ci, w, hc, k1);
#pragma unroll
            for (int a = 0; a < 3; ++a) xi[a] = fmaf(0.5f * hs[a], k1[a], w[a]);
        }
        if (staged) mbar_wait(bar_b, parity);
        if (live) {
            cart_velocity_staged<false>(g, fb, tb, ci, xi, hc, k2);
#pragma unroll
            for (int a = 0; a < 3; ++a) xi[a] = fmaf(0.5f * hs[a], k2[a], w[a]);
            cart_velocity_staged<true>(g, fb, tb, ci, xi, hc, k3);
#pragma unroll
            for (int a = 0; a < 3; ++a) xi[a] = fmaf(hs[a], k3[a], w[a]);
        }
        if (staged) mbar_wait(bar_c, parity);
        if (live) {
            cart_velocity_staged<false>(g, fc, tc, ci, xi, hc, k4);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                float wn = fmaf(hs[a] * (1.0f / 6.0f), (k1[a] + k4[a]) + 2.0f * (k2[a] + k3[a]), w[a]);
                int ifl;
                floor_split<float>(wn, ifl, w[a]);
                ci[a] += ifl;
            }
        }
    }
    if (live) {
        // the block's local frame differs from the stored (never wrapped) cell index by a multiple of n
#pragma unroll
        for (int a = 0; a < 3; ++a) { t.ci[a] = (t.ci[a] & ~(g.n[a] - 1)) + ci[a]; t.w[a] = w[a]; }
        store_record(st + i, t);
    }
}

// ---------------------------------------------------------------------------------------------
// Adams-Bashforth 4 with an RK4 start-up (row f4; "Adams-Bashforth (multi-step)"; reading #31): one
// velocity evaluation per step once three RK4 steps have filled the history.  hist: [n][3][DIM] physical velocities
// f_{n-1}, f_{n-2}, f_{n-3} of each tracer, carried across launches (tracers are not re-bundled in this mode).
template <int DIM, typename TV, typename TC, bool FASTWRAP, bool LD256>
__global__ void __launch_bounds__(256)
cart_ab4_kernel(const __grid_constant__ CartDev g, const PairRec<DIM, TV> *__restrict__ pa, const PairRec<DIM, TV> *__restrict__ pb,
                const PairRec<DIM, TV> *__restrict__ pc, const TC *__restrict__ tau, int nsteps, int first_step, int64_t n,
                CartTracer<DIM, TC> *__restrict__ st, TC *__restrict__ hist, TC hs0, TC hs1, TC hs2)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    CartTracer<DIM, TC> t = load_record(st + i);
    if ((t.meta >> 30) != 0) return;
    const TC hs[3] = {hs0, hs1, hs2};
    int ci[DIM];
    TC w[DIM], h0[DIM], h1[DIM], h2[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        ci[a] = t.ci[a]; w[a] = t.w[a];
        h0[a] = first_step > 0 ? hist[(i * 3 + 0) * DIM + a] : TC(0);
        h1[a] = first_step > 0 ? hist[(i * 3 + 1) * DIM + a] : TC(0);
        h2[a] = first_step > 0 ? hist[(i * 3 + 2) * DIM + a] : TC(0);
    }
    int s = 0;
    bool ok = true;
    for (; s < nsteps; ++s) {
        const TC ta = __ldg(tau + 3 * s), tb = __ldg(tau + 3 * s + 1), tc = __ldg(tau + 3 * s + 2);
        TC k1[DIM], inc[DIM];
        ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pa, ta, ci, w, k1);
        if (!ok) break;
        if (first_step + s < 3) {
            TC k2[DIM], k3[DIM], k4[DIM], xi[DIM];
#pragma unroll
            for (int a = 0; a < DIM; ++a) xi[a] = fma(TC(0.5) * hs[a], k1[a], w[a]);
            ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pb, tb, ci, xi, k2);
            if (!ok) break;
#pragma unroll
            for (int a = 0; a < DIM; ++a) xi[a] = fma(TC(0.5) * hs[a], k2[a], w[a]);
            ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pb, tb, ci, xi, k3);
            if (!ok) break;
#pragma unroll
            for (int a = 0; a < DIM; ++a) xi[a] = fma(hs[a], k3[a], w[a]);
            ok = cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, pc, tc, ci, xi, k4);
            if (!ok) break;
#pragma unroll
            for (int a = 0; a < DIM; ++a) inc[a] = TC(1.0 / 6.0) * ((k1[a] + k4[a]) + TC(2) * (k2[a] + k3[a]));
        } else {
#pragma unroll
            for (int a = 0; a < DIM; ++a)
                inc[a] = TC(1.0 / 24.0) * (((TC(55) * k1[a] - TC(59) * h0[a]) + TC(37) * h1[a]) - TC(9) * h2[a]);
        }
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            int ifl;
            floor_split<TC>(fma(hs[a], inc[a], w[a]), ifl, w[a]);
            ci[a] += ifl;
            h2[a] = h1[a]; h1[a] = h0[a]; h0[a] = k1[a];
        }
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        t.ci[a] = ci[a]; t.w[a] = w[a];
        hist[(i * 3 + 0) * DIM + a] = h0[a]; hist[(i * 3 + 1) * DIM + a] = h1[a]; hist[(i * 3 + 2) * DIM + a] = h2[a];
    }
    if (!ok) t.meta = (1u << 30) | (uint32_t)(first_step + s);
    store_record(st + i, t);
}

// ---------------------------------------------------------------------------------------------
// Split variant (the paper's design: "the RK4 computation was divided into several short
// kernels"; all tracers advance one stage at a time).  One launch per RK4 stage; between the launches the
// stage point (xi) and the running sum k1 + 2 k2 + 2 k3 (acc) live in global memory as [n][DIM] arrays.
// A tracer whose stage point leaves the domain gets its flag at once; its record (position at the start of
// the step) is only rewritten by stage 3 of a step in which all four evaluations succeeded.
template <int DIM, typename TV, typename TC, bool FASTWRAP, bool LD256, int STAGE>
__global__ void __launch_bounds__(256)
cart_stage_kernel(const __grid_constant__ CartDev g, const PairRec<DIM, TV> *__restrict__ rec, TC tau, int step, int64_t n,
                  CartTracer<DIM, TC> *__restrict__ st, TC *__restrict__ xi_g, TC *__restrict__ acc_g, TC hs0, TC hs1, TC hs2)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    CartTracer<DIM, TC> t = load_record(st + i);
    if ((t.meta >> 30) != 0) return;
    const TC hs[3] = {hs0, hs1, hs2};
    TC xi[DIM], k[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) xi[a] = STAGE == 0 ? t.w[a] : xi_g[i * DIM + a];
    if (!cart_velocity<DIM, TV, TC, FASTWRAP, LD256>(g, rec, tau, t.ci, xi, k)) {
        t.meta = (1u << 30) | (uint32_t)step;
        store_record(st + i, t);
        return;
    }
    if constexpr (STAGE < 3) {
        const TC c = STAGE == 2 ? TC(1) : TC(0.5);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            xi_g[i * DIM + a] = fma(c * hs[a], k[a], t.w[a]);
            acc_g[i * DIM + a] = STAGE == 0 ? k[a] : acc_g[i * DIM + a] + TC(2) * k[a];
        }
    } else {
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            TC wn = fma(hs[a] * TC(1.0 / 6.0), acc_g[i * DIM + a] + k[a], t.w[a]);
            int ifl;
            floor_split<TC>(wn, ifl, t.w[a]);
            t.ci[a] += ifl;
        }
        store_record(st + i, t);
    }
}

// ---------------------------------------------------------------------------------------------
// lcs_locate on a Cartesian grid: oracle rule O2 verbatim in fp64 (bit-exact cell ids and weights).
template <int DIM>
__global__ void __launch_bounds__(256) cart_locate_kernel(CartDev g, const double *__restrict__ pos, int64_t n,
                                                           int32_t *__restrict__ cell, double *__restrict__ wout)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int64_t lo[DIM];
    double w[DIM];
    bool inside = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double xi = __dmul_rn(__dsub_rn(pos[i * DIM + a], g.origin[a]), g.inv[a]);
        double f = floor(xi);
        int64_t c = (int64_t)f;
        double wa = __dsub_rn(xi, f);
        int64_t na = g.n[a];
        if (g.periodic[a]) {
            c = ((c % na) + na) % na;
        } else {
            if (!(xi >= 0.0 && xi <= (double)(na - 1))) inside = false;
            if (c == na - 1) { c = na - 2; wa = 1.0; }
        }
        lo[a] = c;
        w[a] = wa;
    }
    if (!inside) {
        cell[i] = -1;
        if (wout) for (int a = 0; a < DIM; ++a) wout[i * DIM + a] = 0.0;
        return;
    }
    int64_t nc0 = g.periodic[0] ? g.n[0] : g.n[0] - 1;
    int64_t nc1 = g.periodic[1] ? g.n[1] : g.n[1] - 1;
    int64_t id = lo[0] + nc0 * lo[1];
    if constexpr (DIM == 3) id += nc0 * nc1 * lo[2];
    cell[i] = (int32_t)id;
    if (wout) for (int a = 0; a < DIM; ++a) wout[i * DIM + a] = w[a];
}

CartDev make_dev(const lcs_field *f)
{
    CartDev g;
    for (int a = 0; a < 3; ++a) {
        g.n[a] = f->cart.n[a]; g.periodic[a] = f->cart.periodic[a]; g.pow2[a] = f->cart.pow2[a];
        g.origin[a] = f->cart.origin[a]; g.spacing[a] = f->cart.spacing[a]; g.inv[a] = f->cart.inv[a];
    }
    g.np0 = f->cart.np[0];
    g.np01 = f->cart.np[0] * f->cart.np[1];
    return g;
}

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// How lcs_advect carves the field's scratch for n tracers and N steps under the current options.  lcs_field_reserve sizes
// the allocation with the same function (worst case over the windows of any [t0, tf]), so the hot call never allocates.
struct CartLayout {
    bool split, ab4, do_bundle, preblend, tma;
    int shift, order, max_fields;
    int64_t nbins, ntiles;
    size_t o_a, o_b, o_xi, o_acc, o_hist, o_tau, o_key, o_cnt, o_tile, o_ftau, o_fields, total;
};

size_t cart_tracer_bytes(const lcs_field *f)
{
    const bool c64 = f->compute_dtype == LCS_F64;
    if (f->dim == 2) return c64 ? sizeof(CartTracer<2, double>) : sizeof(CartTracer<2, float>);
    return c64 ? sizeof(CartTracer<3, double>) : sizeof(CartTracer<3, float>);
}

CartLayout cart_layout(const lcs_field *f, int64_t n, int64_t N)
{
    CartLayout L{};
    const int DIM = f->dim;
    const size_t tcb = lcs_esize(f->compute_dtype), trb = cart_tracer_bytes(f);
    L.split = f->opt_integrator == 2;
    L.ab4 = f->opt_integrator == 3;
    L.do_bundle = !L.ab4 && (f->opt_bundle == 1 || (f->opt_bundle < 0 && n >= (1 << 18)));
    // sort bins: cell index coarsened so that the histogram stays <= 2^24 bins
    int bits = 0;
    for (L.shift = 0;; ++L.shift) {
        bits = 0;
        for (int a = 0; a < DIM; ++a) {
            int cells = ((f->cart.n[a] - 1) >> L.shift) + 1, b = 0;
            while ((1 << b) < cells) ++b;
            bits = b > bits ? b : bits;
        }
        if (bits * DIM <= 24) break;
    }
    L.order = (int)f->opt_bundle_order;               // resolved below once it is known whether the pre-blended integrator runs
    int64_t nkeys = (int64_t)1 << (bits * DIM);
    const bool can_blend = DIM == 3 && f->compute_dtype == LCS_F32 && f->vel_dtype == LCS_F32;
    L.preblend = can_blend && !L.split && !L.ab4 && (f->opt_preblend == 1 || (f->opt_preblend < 0 && n >= (1 << 20)));
    // staged (shared-memory) variant of the pre-blended integrator: periodic power-of-two grids of at most 1024 nodes per axis
    // and at least 4 per axis, tracers bundled in brick order
    bool fastwrap = true;
    for (int a = 0; a < DIM; ++a) fastwrap = fastwrap && f->cart.periodic[a] && f->cart.pow2[a] && f->cart.n[a] <= 1024 && f->cart.n[a] >= 4;
    L.tma = L.preblend && L.do_bundle && f->opt_tma != 0 && fastwrap && L.shift == 0;
    if (L.order < 0) L.order = L.preblend ? 0 : 1;
    if (L.tma && f->opt_tma == 1) L.order = 3;        // tma = 2: staged kernel on the sort order of option bundle_order (experiments)
    if (L.order == 3) {
        if (DIM == 3 && L.shift == 0) nkeys = (int64_t)((f->cart.n[0] + 3) / 4) * ((f->cart.n[1] + 1) / 2) * ((f->cart.n[2] + 1) / 2) * 16;
        else L.order = 1;
    }
    if (L.order == 2) {
        const int64_t sub = (int64_t)((f->cart.n[0] + 1) / 2) * f->cart.n[1] * f->cart.n[2] * 16;
        if (DIM == 3 && L.shift == 0 && sub <= (1 << 24)) nkeys = sub;
        else L.order = 1;
    }
    L.nbins = L.do_bundle ? nkeys + 1 : 0;
    L.ntiles = (L.nbins + bundle::kScanTile - 1) / bundle::kScanTile;
    L.max_fields = L.preblend ? 2 * (int)(f->opt_preblend_steps < N ? f->opt_preblend_steps : N) + 1 : 0;
    size_t off = 0;
    L.o_a = off; off = align_up(off + (size_t)n * trb);
    L.o_b = off; if (L.do_bundle) off = align_up(off + (size_t)n * trb);
    L.o_xi = off; if (L.split) off = align_up(off + (size_t)n * DIM * tcb);
    L.o_acc = off; if (L.split) off = align_up(off + (size_t)n * DIM * tcb);
    L.o_hist = off; if (L.ab4) off = align_up(off + (size_t)n * 3 * DIM * tcb);
    L.o_tau = off; off = align_up(off + (size_t)3 * N * tcb);
    L.o_key = off; if (L.do_bundle) off = align_up(off + (size_t)n * 4);
    L.o_cnt = off; if (L.do_bundle) off = align_up(off + (size_t)L.nbins * 4);
    L.o_tile = off; if (L.do_bundle) off = align_up(off + (size_t)L.ntiles * 4);
    L.o_ftau = off; if (L.preblend) off = align_up(off + ((size_t)3 * N + 8) * 4);
    // one chunk of blended fields, unless resident field sets hold them
    L.o_fields = off; if (L.preblend && f->opt_field_sets == 0) off = align_up(off + (size_t)L.max_fields * (size_t)f->nrec * 32);
    L.total = off;
    return L;
}

template <int DIM, typename TV, typename TC, bool FASTWRAP, bool LD256>
void launch_window(const CartDev &g, const void *const p[3], const TC *d_tau, int first, int count, int64_t n, CartTracer<DIM, TC> *S,
                   const TC *hs, int block, cudaStream_t st)
{
    using Rec = PairRec<DIM, TV>;
    LCS_LAUNCH((cart_window_kernel<DIM, TV, TC, FASTWRAP, LD256>), lcs_blocks(n, block), block, 0, st, g, (const Rec *)p[0], (const Rec *)p[1],
               (const Rec *)p[2], d_tau + 3 * (size_t)first, count, first, n, S, hs[0], hs[1], hs[2]);
}

// one RK4 step of the split variant = 4 launches
template <int DIM, typename TV, typename TC, bool FASTWRAP, bool LD256>
void launch_split_step(const CartDev &g, const void *const p[3], const TC *tau3, int step, int64_t n, CartTracer<DIM, TC> *S, TC *xi,
                       TC *acc, const TC *hs, int block, cudaStream_t st)
{
    using Rec = PairRec<DIM, TV>;
    const unsigned grid = lcs_blocks(n, block);
    LCS_LAUNCH((cart_stage_kernel<DIM, TV, TC, FASTWRAP, LD256, 0>), grid, block, 0, st, g, (const Rec *)p[0], tau3[0], step, n, S, xi, acc, hs[0], hs[1], hs[2]);
    LCS_LAUNCH((cart_stage_kernel<DIM, TV, TC, FASTWRAP, LD256, 1>), grid, block, 0, st, g, (const Rec *)p[1], tau3[1], step, n, S, xi, acc, hs[0], hs[1], hs[2]);
    LCS_LAUNCH((cart_stage_kernel<DIM, TV, TC, FASTWRAP, LD256, 2>), grid, block, 0, st, g, (const Rec *)p[1], tau3[1], step, n, S, xi, acc, hs[0], hs[1], hs[2]);
    LCS_LAUNCH((cart_stage_kernel<DIM, TV, TC, FASTWRAP, LD256, 3>), grid, block, 0, st, g, (const Rec *)p[2], tau3[2], step, n, S, xi, acc, hs[0], hs[1], hs[2]);
}

template <int DIM, typename TV, typename TC>
lcs_status cart_advect_impl(lcs_field *f, int64_t n, const void *seeds_, double t0, double h, int64_t N, void *flowmap_,
                            uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st)
{
    using Tracer = CartTracer<DIM, TC>;
    const TC *seeds = (const TC *)seeds_;
    TC *flowmap = (TC *)flowmap_;
    if (n >= (1LL << 31) || N >= (1LL << 24)) { lcs_set_error("too many seeds or steps for 32-bit tracer records"); return LCS_ERR_INVALID_ARG; }
    std::vector<StepWindow> windows;
    lcs_status rc = lcs_plan_windows(f, t0, h, N, windows);
    if (rc != LCS_OK) return rc;
    const CartLayout L = cart_layout(f, n, N);
    rc = lcs_scratch_check(f, L.total);
    if (rc != LCS_OK) return rc;
    const bool split = L.split, ab4 = L.ab4, do_bundle = L.do_bundle, preblend = L.preblend;
    const int64_t nbins = L.nbins;

    // launch units: a snapshot window is cut into chunks (pre-blended variant: <= preblend_steps steps, whose
    // distinct stage times are blended once per node; otherwise <= bundle_steps steps between re-bundlings)
    constexpr bool kCanBlend = DIM == 3 && sizeof(TC) == 4 && sizeof(TV) == 4;
    struct Unit { int win, first, count, blend, ftau_off, nfields; };
    std::vector<Unit> units;
    std::vector<float> ftau;                          // host copy of the blended stage-time weights: keys of the resident field sets
    for (size_t wi = 0; wi < windows.size(); ++wi) {
        const StepWindow &w = windows[wi];
        const bool blend = preblend && w.s[0] == w.s[1] && w.s[1] == w.s[2];
        int chunk = w.count;
        if (blend) chunk = (int)f->opt_preblend_steps;
        else if (do_bundle && f->opt_bundle_steps > 0) chunk = (int)f->opt_bundle_steps;
        for (int done = 0, cnt = 0; done < w.count; done += cnt) {
            cnt = lcs_early_cut(f, w.first + done, w.count - done < chunk ? w.count - done : chunk);
            Unit u{(int)wi, (int)w.first + done, cnt, blend ? 1 : 0, (int)ftau.size(), 0};
            if (blend) {
                // fields of the chunk: ta_0, tb_0, tc_0 (= ta_1), tb_1, tc_1, ...: 2 count + 1 of them.  tc of a step and ta of
                // the next are the same product t0 + (n + 1) h in the same snapshot pair, hence the same tau bit for bit;
                // should that ever fail, the chunk falls back to pair records.
                bool regular = true;
                for (int s = u.first; s + 1 < u.first + u.count; ++s)
                    regular = regular && (float)lcs_stage_tau(f, t0, h, s, 2, w.s[2]) == (float)lcs_stage_tau(f, t0, h, s + 1, 0, w.s[0]);
                if (regular) {
                    for (int s = u.first; s < u.first + u.count; ++s) {
                        ftau.push_back((float)lcs_stage_tau(f, t0, h, s, 0, w.s[0]));
                        ftau.push_back((float)lcs_stage_tau(f, t0, h, s, 1, w.s[1]));
                    }
                    ftau.push_back((float)lcs_stage_tau(f, t0, h, u.first + u.count - 1, 2, w.s[2]));
                    u.nfields = 2 * u.count + 1;
                } else {
                    u.blend = 0;
                }
            }
            units.push_back(u);
        }
    }

    char *base = (char *)f->scratch.buf;
    Tracer *cur = (Tracer *)(base + L.o_a), *alt = (Tracer *)(base + L.o_b);
    TC *d_xi = (TC *)(base + L.o_xi), *d_acc = (TC *)(base + L.o_acc), *d_tau = (TC *)(base + L.o_tau);
    uint32_t *d_key = (uint32_t *)(base + L.o_key), *d_cnt = (uint32_t *)(base + L.o_cnt), *d_tile = (uint32_t *)(base + L.o_tile);
    float *d_ftau = (float *)(base + L.o_ftau);

    CartDev g = make_dev(f);
    const int block = f->opt_block ? (int)(f->opt_block > 256 ? 256 : f->opt_block) : 256;
    LCS_LAUNCH((cart_init_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, g, seeds, n, cur);
    bool fast = true;
    for (int a = 0; a < DIM; ++a) fast = fast && g.periodic[a] && g.pow2[a];
    const bool ld256 = f->opt_ld256 != 0;
    TC hs[3] = {TC(1), TC(1), TC(1)};
    for (int a = 0; a < DIM; ++a) hs[a] = (TC)(h * f->cart.inv[a]);
    const int dir = h > 0 ? 1 : -1;

    auto rebundle = [&]() -> lcs_status {
        LCS_CUDA_OK(cudaMemsetAsync(d_cnt, 0, (size_t)nbins * 4, st));
        LCS_LAUNCH((cart_key_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, g, cur, n, L.shift, L.order, (uint32_t)(nbins - 1), d_key, d_cnt);
        bundle::sort_records<Tracer>(cur, alt, d_key, d_cnt, d_tile, n, nbins, st);
        std::swap(cur, alt);
        return LCS_OK;
    };

    // row f1: at an evaluation point, scatter positions and flags to the caller's order and evaluate C for complete stencils
    auto early_eval = [&](int64_t end) -> lcs_status {
        if (!lcs_early_due(f, end, N)) return LCS_OK;
        LCS_LAUNCH((cart_final_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, g, seeds, n, cur, (int32_t)N, (TC *)f->early.flowmap, f->early.flag,
                   (int32_t *)nullptr);
        return lcs_early_cg_eval(f, end, st);
    };
    int cur_win = -1, since_bundle = 0;
    const void *p[3] = {nullptr, nullptr, nullptr}, *raw_a = nullptr, *raw_b = nullptr;
    for (size_t ui = 0; ui < units.size(); ++ui) {
        const Unit &u = units[ui];
        const StepWindow &w = windows[u.win];
        const bool new_win = u.win != cur_win;
        if (new_win) {
            // what the units of this window gather from: raw snapshots (blended chunks) and / or pair records
            bool need_raw = false, need_pairs = false;
            for (size_t uj = ui; uj < units.size() && units[uj].win == u.win; ++uj) (units[uj].blend ? need_raw : need_pairs) = true;
            if (need_raw) {
                rc = lcs_field_acquire_raw(f, w.s[0], st, &raw_a, &raw_b);
                if (rc != LCS_OK) return rc;
            }
            if (need_pairs) {
                for (int k = 0; k < 3; ++k) {
                    rc = lcs_field_require_pair(f, w.s[k], st, &p[k]);
                    if (rc != LCS_OK) return rc;
                }
                // stage-time weights of the window's steps, computed on the device (no host-to-device copy in the hot call)
                rc = lcs_fill_stage_tau(f, t0, h, w.first, w.count, w.s, d_tau, nullptr, st);
                if (rc != LCS_OK) return rc;
            }
            // stream the snapshot the NEXT window will need while this one computes (side stream)
            lcs_field_prefetch(f, dir > 0 ? w.s[2] + 2 : w.s[2] - 1, w.s[2], w.s[2] + 1);
            cur_win = u.win;
            f->info_windows++;
        }
        if (do_bundle && (new_win || (f->opt_bundle_steps > 0 && since_bundle >= f->opt_bundle_steps))) {
            rc = rebundle();
            if (rc != LCS_OK) return rc;
            since_bundle = 0;
        }
        since_bundle += u.count;
        if constexpr (kCanBlend) {
            if (u.blend) {
                XPair *fields = (XPair *)(base + L.o_fields);
                bool need_blend = true;
                FieldSet *filling = nullptr;
                const float *tb = ftau.data() + u.ftau_off;
                if (f->opt_field_sets > 0) {
                    // resident field sets (allocated by lcs_field_reserve): reuse the set blended from the same snapshot pair
                    // for the same stage times, else blend into the least recently used one
                    const size_t bytes = (size_t)u.nfields * (size_t)f->nrec * 32;
                    FieldSet *hit = nullptr, *victim = nullptr;
                    for (FieldSet &fs : f->field_sets)
                        if (fs.buf && fs.pair == w.s[0] && fs.tau.size() == (size_t)u.nfields && std::equal(fs.tau.begin(), fs.tau.end(), tb)) hit = &fs;
                    if (!hit) {
                        for (FieldSet &fs : f->field_sets) if (fs.buf && fs.bytes >= bytes && (!victim || fs.age < victim->age)) victim = &fs;
                        if (!victim) {
                            lcs_set_error("no resident field set of %zu bytes is reserved: call lcs_field_reserve after setting field_sets", bytes);
                            return LCS_ERR_OOM;
                        }
                        victim->pair = -1;                           // the old key dies BEFORE the buffer is overwritten;
                        victim->tau.clear();                         // the new one is set once the blend is enqueued
                        f->info_field_set_misses++;
                        hit = filling = victim;
                    } else {
                        need_blend = false;
                        f->info_field_set_hits++;
                    }
                    hit->age = ++f->field_set_clock;
                    fields = (XPair *)hit->buf;
                }
                if (need_blend) {
                    rc = lcs_fill_stage_tau(f, t0, h, u.first, u.count, w.s, nullptr, d_ftau + u.ftau_off, st);
                    if (rc != LCS_OK) return rc;
                    LCS_LAUNCH(blend_xpair_kernel, lcs_blocks(f->nrec, 256), 256, 0, st, (const float *)raw_a, (const float *)raw_b, g.n[0],
                               g.n[1], g.n[2], f->cart.np[0], f->cart.np[1], f->cart.np[2], d_ftau + u.ftau_off, u.nfields, fields, f->nrec);
                    LCS_CUDA_OK(cudaGetLastError());
                    if (filling) { filling->pair = w.s[0]; filling->tau.assign(tb, tb + u.nfields); }
                }
                {
                    WindowTimer timer(f, st);
                    if (L.tma) {
                        const int cap = (int)f->opt_tma_cap;
                        const size_t smem = (size_t)cap * 64 + 16 + 3 * 8 * sizeof(int);
                        LCS_LAUNCH(cart_xpair_tma_kernel, lcs_blocks(n, kStageBlock), kStageBlock, smem, st, g, (const XPair *)fields, f->nrec, u.count,
                                   u.first, n, cur, hs[0], hs[1], hs[2], cap);
                    } else if (fast)
                        LCS_LAUNCH((cart_xpair_kernel<true, false>), lcs_blocks(n, block), block, 0, st, g, (const XPair *)fields, f->nrec,
                                   u.count, u.first, n, cur, hs[0], hs[1], hs[2], SeriesTail{});
                    else
                        LCS_LAUNCH((cart_xpair_kernel<false, false>), lcs_blocks(n, block), block, 0, st, g, (const XPair *)fields, f->nrec,
                                   u.count, u.first, n, cur, hs[0], hs[1], hs[2], SeriesTail{});
                }
                bool last_blend_of_win = true;
                for (size_t uj = ui + 1; uj < units.size() && units[uj].win == u.win; ++uj) last_blend_of_win = last_blend_of_win && !units[uj].blend;
                if (last_blend_of_win) { rc = lcs_field_release_raw(f, w.s[0], st); if (rc != LCS_OK) return rc; }
                rc = early_eval((int64_t)u.first + u.count);
                if (rc != LCS_OK) return rc;
                continue;
            }
        }
        WindowTimer timer(f, st);
        if (ab4) {
            using Rec = PairRec<DIM, TV>;
            TC *d_hist = (TC *)(base + L.o_hist);
#define LCS_AB4(FW, LD) LCS_LAUNCH((cart_ab4_kernel<DIM, TV, TC, FW, LD>), lcs_blocks(n, block), block, 0, st, g, (const Rec *)p[0], (const Rec *)p[1], \
                                   (const Rec *)p[2], d_tau + 3 * (size_t)u.first, u.count, u.first, n, cur, d_hist, hs[0], hs[1], hs[2])
            if (fast && ld256) LCS_AB4(true, true);
            else if (fast) LCS_AB4(true, false);
            else if (ld256) LCS_AB4(false, true);
            else LCS_AB4(false, false);
#undef LCS_AB4
        } else if (!split) {
            if (fast && ld256) launch_window<DIM, TV, TC, true, true>(g, p, d_tau, u.first, u.count, n, cur, hs, block, st);
            else if (fast) launch_window<DIM, TV, TC, true, false>(g, p, d_tau, u.first, u.count, n, cur, hs, block, st);
            else if (ld256) launch_window<DIM, TV, TC, false, true>(g, p, d_tau, u.first, u.count, n, cur, hs, block, st);
            else launch_window<DIM, TV, TC, false, false>(g, p, d_tau, u.first, u.count, n, cur, hs, block, st);
        } else {
            for (int s = u.first; s < u.first + u.count; ++s) {
                const TC t3[3] = {(TC)lcs_stage_tau(f, t0, h, s, 0, w.s[0]), (TC)lcs_stage_tau(f, t0, h, s, 1, w.s[1]),
                                  (TC)lcs_stage_tau(f, t0, h, s, 2, w.s[2])};
                if (fast && ld256) launch_split_step<DIM, TV, TC, true, true>(g, p, t3, s, n, cur, d_xi, d_acc, hs, block, st);
                else if (fast) launch_split_step<DIM, TV, TC, true, false>(g, p, t3, s, n, cur, d_xi, d_acc, hs, block, st);
                else if (ld256) launch_split_step<DIM, TV, TC, false, true>(g, p, t3, s, n, cur, d_xi, d_acc, hs, block, st);
                else launch_split_step<DIM, TV, TC, false, false>(g, p, t3, s, n, cur, d_xi, d_acc, hs, block, st);
            }
        }
        rc = early_eval((int64_t)u.first + u.count);
        if (rc != LCS_OK) return rc;
    }
    LCS_LAUNCH((cart_final_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, g, seeds, n, cur, (int32_t)N, flowmap, exit_flag, exit_step);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
// FTLE time series (BASELINE.json config 5; a sequence of seed grids released one after the other through the
// same data).  Volumes whose integration intervals overlap are advanced TOGETHER: the tracers of every volume that is inside a
// snapshot window are bundled into one set, so that one blend of the window's stage-time fields and one integrator launch serve
// them all, at 8-30 tracers per cell instead of 3 (the gathers of a warp then fall into a handful of 128-byte lines: 64 -> 76 G
// seed-steps/s inside the kernel).  A volume joins the set when its release time is reached (cart_init_kernel
// appends its records) and leaves it after its last step (cart_final_series_kernel writes its outputs and marks its records dead;
// the next re-bundling drops them).  Records carry their own step count (per_tracer_steps).
// Batching needs volumes that are the same integration shifted by whole snapshot intervals, on the pre-blended bundled path;
// anything else is integrated volume by volume (plan.batched == false).
struct SeriesPlan {
    bool batched = false;
    struct Unit { int pair, first, count, ftau_off, nfields, chunk; };
    std::vector<Unit> units;                 // launch units of ONE volume (pair = snapshot pair of volume 0, chunk = index inside its window)
    std::vector<float> ftau;
    std::vector<int> shift;                  // volume k uses pair + shift[k]
    struct Layer { int pair, chunk, unit; std::vector<int> start_vols, finish_vols; };   // unit = a member's unit (all members share count and stage times)
    std::vector<Layer> layers;               // in integration order
    int64_t cap_records = 0;                 // largest number of records in the set (incl. those dropped by the next re-bundling)
};

lcs_status series_plan(const lcs_field *f, int64_t n, int n_vol, const double *t_start, double h, int64_t N, SeriesPlan &P)
{
    P = SeriesPlan();
    const CartLayout L1 = cart_layout(f, n * (int64_t)std::min(n_vol, 2), N);
    if (!L1.preblend || !L1.do_bundle || L1.tma || n_vol < 2) return LCS_OK;
    std::vector<StepWindow> w0;
    lcs_status rc = lcs_plan_windows(f, t_start[0], h, N, w0);
    if (rc != LCS_OK) return rc;
    // units of volume 0 (as in cart_advect_impl: a window is cut into chunks of preblend_steps steps)
    for (const StepWindow &w : w0) {
        if (!(w.s[0] == w.s[1] && w.s[1] == w.s[2])) return LCS_OK;
        const int chunk = (int)f->opt_preblend_steps;
        for (int done = 0, cnt = 0, ci = 0; done < w.count; done += cnt, ++ci) {
            cnt = w.count - done < chunk ? w.count - done : chunk;
            SeriesPlan::Unit u{w.s[0], (int)w.first + done, cnt, (int)P.ftau.size(), 2 * cnt + 1, ci};
            for (int s = u.first; s + 1 < u.first + u.count; ++s)
                if ((float)lcs_stage_tau(f, t_start[0], h, s, 2, w.s[2]) != (float)lcs_stage_tau(f, t_start[0], h, s + 1, 0, w.s[0])) return LCS_OK;
            for (int s = u.first; s < u.first + u.count; ++s) {
                P.ftau.push_back((float)lcs_stage_tau(f, t_start[0], h, s, 0, w.s[0]));
                P.ftau.push_back((float)lcs_stage_tau(f, t_start[0], h, s, 1, w.s[1]));
            }
            P.ftau.push_back((float)lcs_stage_tau(f, t_start[0], h, u.first + u.count - 1, 2, w.s[2]));
            P.units.push_back(u);
        }
    }
    // every other volume: the same units in snapshot pairs shifted by a constant, with the same stage-time weights bit for bit
    P.shift.assign(n_vol, 0);
    for (int k = 1; k < n_vol; ++k) {
        std::vector<StepWindow> wk;
        rc = lcs_plan_windows(f, t_start[k], h, N, wk);
        if (rc != LCS_OK) return rc;
        if (wk.size() != w0.size()) return LCS_OK;
        const int sh = wk[0].s[0] - w0[0].s[0];
        for (size_t i = 0; i < wk.size(); ++i)
            if (wk[i].first != w0[i].first || wk[i].count != w0[i].count || wk[i].s[0] != w0[i].s[0] + sh || wk[i].s[1] != wk[i].s[0] ||
                wk[i].s[2] != wk[i].s[0]) return LCS_OK;
        for (const SeriesPlan::Unit &u : P.units) {
            const float *tb = P.ftau.data() + u.ftau_off;
            for (int s = u.first, j = 0; s < u.first + u.count; ++s, j += 2)
                if ((float)lcs_stage_tau(f, t_start[k], h, s, 0, u.pair + sh) != tb[j] || (float)lcs_stage_tau(f, t_start[k], h, s, 1, u.pair + sh) != tb[j + 1]) return LCS_OK;
            if ((float)lcs_stage_tau(f, t_start[k], h, u.first + u.count - 1, 2, u.pair + sh) != tb[2 * u.count]) return LCS_OK;
        }
        P.shift[k] = sh;
    }
    // layers: (snapshot pair, chunk inside the window) in integration order; volume k runs its unit i in layer
    // (units[i].pair + shift[k], units[i].chunk).  Units that meet in a layer must be the same steps of the window: same count and
    // the same stage-time weights bit for bit (they belong to different unit indices of volume 0's table).
    const int dir = h > 0 ? 1 : -1;
    const int last = (int)P.units.size() - 1;
    struct Ev { int64_t order; int pair, unit, vol; };
    std::vector<Ev> evs;
    for (int k = 0; k < n_vol; ++k)
        for (size_t i = 0; i < P.units.size(); ++i)
            evs.push_back({(int64_t)dir * (P.units[i].pair + P.shift[k]) * 65536 + (int64_t)P.units[i].chunk, P.units[i].pair + P.shift[k], (int)i, k});
    std::sort(evs.begin(), evs.end(), [](const Ev &a, const Ev &b) { return a.order != b.order ? a.order < b.order : a.vol < b.vol; });
    for (const Ev &e : evs) {
        const SeriesPlan::Unit &u = P.units[e.unit];
        if (P.layers.empty() || P.layers.back().pair != e.pair || P.layers.back().chunk != u.chunk) P.layers.push_back({e.pair, u.chunk, e.unit, {}, {}});
        SeriesPlan::Layer &ly = P.layers.back();
        const SeriesPlan::Unit &r = P.units[ly.unit];
        if (r.count != u.count || !std::equal(P.ftau.begin() + r.ftau_off, P.ftau.begin() + r.ftau_off + r.nfields, P.ftau.begin() + u.ftau_off)) {
            P.layers.clear();
            return LCS_OK;
        }
        if (e.unit == 0) ly.start_vols.push_back(e.vol);
        if (e.unit == last) ly.finish_vols.push_back(e.vol);
    }
    // largest record count: live volumes + those that finished in the previous layer (dropped by this layer's re-bundling)
    int64_t act = 0, finished_prev = 0;
    for (const SeriesPlan::Layer &ly : P.layers) {
        act += (int64_t)ly.start_vols.size();
        P.cap_records = std::max(P.cap_records, act * n);
        act -= finished_prev;
        finished_prev = (int64_t)ly.finish_vols.size();
    }
    P.batched = true;
    return LCS_OK;
}

lcs_status cart_advect_series_batched(lcs_field *f, const SeriesPlan &P, int64_t n, const float *seeds, int n_vol, double t0_first, double h, int64_t N,
                                      float *flowmaps, uint8_t *exit_flags, int32_t *exit_steps, cudaStream_t st)
{
    using Tracer = CartTracer<3, float>;
    const CartLayout L = cart_layout(f, P.cap_records, N);
    lcs_status rc = lcs_scratch_check(f, L.total);
    if (rc != LCS_OK) return rc;
    char *base = (char *)f->scratch.buf;
    Tracer *cur = (Tracer *)(base + L.o_a), *alt = (Tracer *)(base + L.o_b);
    uint32_t *d_key = (uint32_t *)(base + L.o_key), *d_cnt = (uint32_t *)(base + L.o_cnt), *d_tile = (uint32_t *)(base + L.o_tile);
    float *d_ftau = (float *)(base + L.o_ftau);
    XPair *fields = (XPair *)(base + L.o_fields);
    if (f->opt_field_sets > 0) { lcs_set_error("lcs_advect_series blends every window once and takes no resident field sets: set field_sets = 0"); return LCS_ERR_INVALID_ARG; }
    CartDev g = make_dev(f);
    const int block = f->opt_block ? (int)(f->opt_block > 256 ? 256 : f->opt_block) : 256;
    bool fast = true;
    for (int a = 0; a < 3; ++a) fast = fast && g.periodic[a] && g.pow2[a];
    float hs[3];
    for (int a = 0; a < 3; ++a) hs[a] = (float)(h * f->cart.inv[a]);
    const int dir = h > 0 ? 1 : -1;
    int64_t n_act = 0;
    std::vector<int> to_finish;
    int cur_pair = -1;
    const void *raw_a = nullptr, *raw_b = nullptr;
    auto finalize = [&](const std::vector<int> &vols) -> lcs_status {
        for (int k : vols)
            LCS_LAUNCH((cart_final_series_kernel<3, float>), lcs_blocks(n_act, 256), 256, 0, st, g, seeds, n_act, cur, (int32_t)(k * n), (int32_t)((k + 1) * n),
                       (int32_t)N, flowmaps, exit_flags, exit_steps);
        LCS_CUDA_OK(cudaGetLastError());
        return LCS_OK;
    };
    // fused bookkeeping (the usual series: at most one volume finishes per layer): the integrator leaves every record's sort key
    // for the next re-bundling and writes the outputs of the finishing volume itself; otherwise a key kernel per layer and a scan of
    // the set per finished volume
    bool fused = true;
    for (const SeriesPlan::Layer &ly : P.layers) fused = fused && ly.finish_vols.size() <= 1;
    const KeyOut ko{d_key, d_cnt, L.shift, L.order, (uint32_t)(L.nbins - 1)};
    if (fused) LCS_CUDA_OK(cudaMemsetAsync(d_cnt, 0, (size_t)L.nbins * 4, st));
    for (size_t li = 0; li < P.layers.size(); ++li) {
        const SeriesPlan::Layer &ly = P.layers[li];
        const SeriesPlan::Unit &u = P.units[ly.unit];
        // volumes that completed their last unit in the previous layer leave; volumes whose first unit this is join
        int64_t dropped = 0;
        if (!fused) {
            rc = finalize(to_finish);
            if (rc != LCS_OK) return rc;
            dropped = (int64_t)to_finish.size() * n;
            to_finish.clear();
        } else if (li > 0) {
            dropped = (int64_t)P.layers[li - 1].finish_vols.size() * n;
        }
        for (int k : ly.start_vols) {
            KeyOut kn = ko;
            kn.key = fused ? d_key + n_act : nullptr;
            LCS_LAUNCH((cart_init_kernel<3, float>), lcs_blocks(n, 256), 256, 0, st, g, seeds, n, cur + n_act, (int32_t)(k * n), kn);
            n_act += n;
        }
        // re-bundle the whole set (drops the dead records)
        if (!fused) {
            LCS_CUDA_OK(cudaMemsetAsync(d_cnt, 0, (size_t)L.nbins * 4, st));
            LCS_LAUNCH((cart_key_kernel<3, float>), lcs_blocks(n_act, 256), 256, 0, st, g, cur, n_act, L.shift, L.order, (uint32_t)(L.nbins - 1), d_key, d_cnt);
        }
        bundle::sort_records<Tracer>(cur, alt, d_key, d_cnt, d_tile, n_act, L.nbins, st);
        std::swap(cur, alt);
        n_act -= dropped;
        if (fused) LCS_CUDA_OK(cudaMemsetAsync(d_cnt, 0, (size_t)L.nbins * 4, st));      // histogram of the NEXT re-bundling
        if (ly.pair != cur_pair) {
            if (cur_pair >= 0) { rc = lcs_field_release_raw(f, cur_pair, st); if (rc != LCS_OK) return rc; }
            rc = lcs_field_acquire_raw(f, ly.pair, st, &raw_a, &raw_b);
            if (rc != LCS_OK) return rc;
            lcs_field_prefetch(f, dir > 0 ? ly.pair + 2 : ly.pair - 1, ly.pair, ly.pair + 1);
            cur_pair = ly.pair;
            f->info_windows++;
        }
        // the stage-time weights of the unit are those of volume 0's copy of it (identical for every volume: series_plan checked)
        {
            const int32_t s3[3] = {u.pair, u.pair, u.pair};
            rc = lcs_fill_stage_tau(f, t0_first, h, u.first, u.count, s3, nullptr, d_ftau, st);
            if (rc != LCS_OK) return rc;
        }
        LCS_LAUNCH(blend_xpair_kernel, lcs_blocks(f->nrec, 256), 256, 0, st, (const float *)raw_a, (const float *)raw_b, g.n[0], g.n[1], g.n[2],
                   f->cart.np[0], f->cart.np[1], f->cart.np[2], d_ftau, u.nfields, fields, f->nrec);
        SeriesTail sr{};
        sr.N = (int32_t)N;
        if (fused) {
            sr.ko = ko;
            sr.fin_lo = sr.fin_hi = 0;
            if (!ly.finish_vols.empty()) { sr.fin_lo = (int32_t)(ly.finish_vols[0] * n); sr.fin_hi = (int32_t)((ly.finish_vols[0] + 1) * n); }
            sr.seeds = seeds; sr.flowmap = flowmaps; sr.exit_flag = exit_flags; sr.exit_step = exit_steps;
        }
        {
            WindowTimer timer(f, st);
            if (fast)
                LCS_LAUNCH((cart_xpair_kernel<true, true>), lcs_blocks(n_act, block), block, 0, st, g, (const XPair *)fields, f->nrec, u.count, 0, n_act, cur,
                           hs[0], hs[1], hs[2], sr);
            else
                LCS_LAUNCH((cart_xpair_kernel<false, true>), lcs_blocks(n_act, block), block, 0, st, g, (const XPair *)fields, f->nrec, u.count, 0, n_act, cur,
                           hs[0], hs[1], hs[2], sr);
        }
        LCS_CUDA_OK(cudaGetLastError());
        if (!fused) to_finish = ly.finish_vols;
    }
    rc = finalize(to_finish);
    if (rc != LCS_OK) return rc;
    if (cur_pair >= 0) { rc = lcs_field_release_raw(f, cur_pair, st); if (rc != LCS_OK) return rc; }
    (void)n_vol;
    f->info_series_layers = (int64_t)P.layers.size();
    return LCS_OK;
}

}  // namespace

size_t lcs_cart_scratch_bytes(const lcs_field *f, int64_t n, int64_t N) { return cart_layout(f, n, N).total; }

lcs_status lcs_cart_tma_configure(lcs_field *f)
{
    const size_t smem = (size_t)f->opt_tma_cap * 64 + 16 + 3 * 8 * sizeof(int);
    if (smem > 48 * 1024) LCS_CUDA_OK(cudaFuncSetAttribute(cart_xpair_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    return LCS_OK;
}

size_t lcs_cart_field_set_bytes(const lcs_field *f, int64_t N)
{
    const CartLayout L = cart_layout(f, (int64_t)1 << 20, N);      // sets are used by the pre-blended integrator only
    return (f->opt_preblend != 0 && L.max_fields > 0) ? (size_t)L.max_fields * (size_t)f->nrec * 32 : 0;
}

// lcs_advect_series on a Cartesian grid: batched when series_plan allows it, else volume by volume
lcs_status lcs_cart_advect_series(lcs_field *f, int64_t n, const void *seeds, int n_vol, const double *t_start, double h, int64_t N,
                                  void *flowmaps, uint8_t *exit_flags, int32_t *exit_steps, cudaStream_t st, int64_t *cap_records_out)
{
    SeriesPlan P;
    lcs_status rc = series_plan(f, n, n_vol, t_start, h, N, P);
    if (rc != LCS_OK) return rc;
    if (n_vol * n >= (1LL << 31)) { lcs_set_error("n_vol * n must stay below 2^31"); return LCS_ERR_INVALID_ARG; }
    if (cap_records_out) { *cap_records_out = P.batched ? P.cap_records : n; return LCS_OK; }      // planning only (lcs_advect_series_reserve)
    f->info_series_layers = 0;
    if (P.batched)
        return cart_advect_series_batched(f, P, n, (const float *)seeds, n_vol, t_start[0], h, N, (float *)flowmaps, exit_flags, exit_steps, st);
    const size_t es = lcs_esize(f->compute_dtype);
    for (int k = 0; k < n_vol; ++k) {
        rc = lcs_cart_advect(f, n, seeds, t_start[k], h, N, (char *)flowmaps + (size_t)k * n * f->dim * es, exit_flags ? exit_flags + (size_t)k * n : nullptr,
                             exit_steps ? exit_steps + (size_t)k * n : nullptr, st);
        if (rc != LCS_OK) return rc;
    }
    return LCS_OK;
}

lcs_status lcs_cart_locate(lcs_field *f, int64_t n, const double *pos, int32_t *cell, double *w, cudaStream_t st)
{
    CartDev g = make_dev(f);
    if (f->dim == 2) LCS_LAUNCH((cart_locate_kernel<2>), lcs_blocks(n, 256), 256, 0, st, g, pos, n, cell, w);
    else LCS_LAUNCH((cart_locate_kernel<3>), lcs_blocks(n, 256), 256, 0, st, g, pos, n, cell, w);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

lcs_status lcs_cart_advect(lcs_field *f, int64_t n, const void *seeds, double t0, double h, int64_t N, void *flowmap,
                           uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st)
{
    const bool v64 = f->vel_dtype == LCS_F64, c64 = f->compute_dtype == LCS_F64;
    if (f->dim == 2) {
        if (c64) return cart_advect_impl<2, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64) return cart_advect_impl<2, float, float>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    } else {
        if (c64) return cart_advect_impl<3, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64) return cart_advect_impl<3, float, float>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    }
    lcs_set_error("fp64 velocity with fp32 arithmetic is not supported (compute_dtype must be >= vel_dtype)");
    return LCS_ERR_INVALID_ARG;
}
