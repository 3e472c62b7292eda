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
//  * gathers read "pair records" {a, b-a}: both time levels of a node in one 32-byte sector, the time
//    blend is one FMA per component.
//  * fused variant: one thread runs every RK4 step of a snapshot window; split variant (the paper's): one
//    short kernel per RK4 stage with the tracer state in global memory.
#include <math.h>

#include "lcs_internal.cuh"

namespace {

struct CartDev {
    int n[3];
    int periodic[3];
    int pow2[3];
    double origin[3], spacing[3], inv[3];
};

template <typename TC> struct CartState {
    int32_t *ci[3];
    TC *w[3];
    int32_t *steps;
    uint8_t *flag;
};

template <typename T> struct Vec2 {};
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

// time-blended velocity at one node: out = a + tau * d  (one FMA per component)
template <int DIM, typename TV, typename TC>
__device__ __forceinline__ void node_velocity(const PairRec<DIM, TV> *__restrict__ rec, int64_t node, TC tau, TC *out)
{
    if constexpr (DIM == 3 && sizeof(TV) == 4) {
        const float4 *p = reinterpret_cast<const float4 *>(rec + node);
        float4 a = __ldg(p), d = __ldg(p + 1);
        out[0] = fma(tau, (TC)d.x, (TC)a.x);
        out[1] = fma(tau, (TC)d.y, (TC)a.y);
        out[2] = fma(tau, (TC)d.z, (TC)a.z);
    } else if constexpr (DIM == 3) {
        const double2 *p = reinterpret_cast<const double2 *>(rec + node);
        double2 a0 = __ldg(p), a1 = __ldg(p + 1), d0 = __ldg(p + 2), d1 = __ldg(p + 3);
        out[0] = fma(tau, (TC)d0.x, (TC)a0.x);
        out[1] = fma(tau, (TC)d0.y, (TC)a0.y);
        out[2] = fma(tau, (TC)d1.x, (TC)a1.x);
    } else if constexpr (sizeof(TV) == 8) {
        const double2 *p = reinterpret_cast<const double2 *>(rec + node);
        double2 a = __ldg(p), d = __ldg(p + 1);
        out[0] = fma(tau, (TC)d.x, (TC)a.x);
        out[1] = fma(tau, (TC)d.y, (TC)a.y);
    } else {
        float4 r = __ldg(reinterpret_cast<const float4 *>(rec + node));
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

// u(x,t) at the point (ci + xi) in grid units, xi = offset relative to the tracer's cell (any magnitude).
// Returns false if the point is outside a non-periodic axis (closed upper end, as in oracle rule O2).
template <int DIM, typename TV, typename TC, bool FASTWRAP>
__device__ __forceinline__ bool cart_velocity(const CartDev &g, const PairRec<DIM, TV> *__restrict__ rec, TC tau,
                                              const int *ci, const TC *xi, TC *u)
{
    int lo[DIM], hi[DIM];
    TC wl[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        TC fl = floor(xi[a]);
        wl[a] = xi[a] - fl;
        int c = ci[a] + (int)fl;
        if constexpr (FASTWRAP) {
            lo[a] = c & (g.n[a] - 1);
            hi[a] = (c + 1) & (g.n[a] - 1);
        } else if (g.periodic[a]) {
            lo[a] = wrap_index(c, g.n[a], g.pow2[a]);
            hi[a] = lo[a] + 1 == g.n[a] ? 0 : lo[a] + 1;
        } else {
            if (c == g.n[a] - 1 && wl[a] == TC(0)) { c = g.n[a] - 2; wl[a] = TC(1); }
            if (c < 0 || c > g.n[a] - 2) return false;
            lo[a] = c;
            hi[a] = c + 1;
        }
    }
    if constexpr (DIM == 2) {
        int64_t r0 = (int64_t)lo[1] * g.n[0], r1 = (int64_t)hi[1] * g.n[0];
        TC v00[2], v10[2], v01[2], v11[2];
        node_velocity<2, TV, TC>(rec, r0 + lo[0], tau, v00);
        node_velocity<2, TV, TC>(rec, r0 + hi[0], tau, v10);
        node_velocity<2, TV, TC>(rec, r1 + lo[0], tau, v01);
        node_velocity<2, TV, TC>(rec, r1 + hi[0], tau, v11);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            TC a0 = fma(wl[0], v10[c] - v00[c], v00[c]);
            TC a1 = fma(wl[0], v11[c] - v01[c], v01[c]);
            u[c] = fma(wl[1], a1 - a0, a0);
        }
    } else {
        int64_t n0 = g.n[0], n01 = (int64_t)g.n[0] * g.n[1];
        int64_t r00 = lo[1] * n0 + lo[2] * n01, r10 = hi[1] * n0 + lo[2] * n01;
        int64_t r01 = lo[1] * n0 + hi[2] * n01, r11 = hi[1] * n0 + hi[2] * n01;
        TC v[8][3];
        node_velocity<3, TV, TC>(rec, r00 + lo[0], tau, v[0]);
        node_velocity<3, TV, TC>(rec, r00 + hi[0], tau, v[1]);
        node_velocity<3, TV, TC>(rec, r10 + lo[0], tau, v[2]);
        node_velocity<3, TV, TC>(rec, r10 + hi[0], tau, v[3]);
        node_velocity<3, TV, TC>(rec, r01 + lo[0], tau, v[4]);
        node_velocity<3, TV, TC>(rec, r01 + hi[0], tau, v[5]);
        node_velocity<3, TV, TC>(rec, r11 + lo[0], tau, v[6]);
        node_velocity<3, TV, TC>(rec, r11 + hi[0], tau, v[7]);
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
template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cart_init_kernel(CartDev g, const TC *__restrict__ seeds, int64_t n, CartState<TC> st)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint8_t fl = 0;
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
        st.ci[a][i] = c;
        st.w[a][i] = (TC)w;
    }
    st.flag[i] = fl;
    st.steps[i] = 0;
}

// (cell, offset) -> physical flow map + flags
template <int DIM, typename TC>
__global__ void __launch_bounds__(256) cart_final_kernel(CartDev g, const TC *__restrict__ seeds, int64_t n, CartState<TC> st,
                                                          int32_t N, TC *__restrict__ flowmap, uint8_t *__restrict__ exit_flag,
                                                          int32_t *__restrict__ exit_step)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint8_t fl = st.flag[i];
    TC out[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        if (fl == 2) out[a] = seeds[i * DIM + a];
        else out[a] = (TC)(g.origin[a] + ((double)st.ci[a][i] + (double)st.w[a][i]) * g.spacing[a]);
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) flowmap[i * DIM + a] = out[a];
    if (exit_flag) exit_flag[i] = fl;
    if (exit_step) exit_step[i] = fl == 0 ? N : (fl == 2 ? 0 : st.steps[i]);
}

// ---------------------------------------------------------------------------------------------
// Fused variant: one thread = one tracer, every RK4 step of the window.  hs[a] = h / spacing[a] turns a
// physical velocity into cells per step.  tau: [nsteps][3] time weights of (ta, tb, tc).
template <int DIM, typename TV, typename TC, bool FASTWRAP>
__global__ void __launch_bounds__(256)
cart_window_kernel(const __grid_constant__ CartDev g, const PairRec<DIM, TV> *__restrict__ pa,
                   const PairRec<DIM, TV> *__restrict__ pb, const PairRec<DIM, TV> *__restrict__ pc,
                   const TC *__restrict__ tau, int nsteps, int first_step, int64_t n, CartState<TC> st, TC hs0, TC hs1, TC hs2)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (st.flag[i] != 0) return;
    const TC hs[3] = {hs0, hs1, hs2};
    int ci[DIM];
    TC w[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) { ci[a] = st.ci[a][i]; w[a] = st.w[a][i]; }
    int s = 0;
    bool ok = true;
    for (; s < nsteps; ++s) {
        const TC ta = __ldg(tau + 3 * s), tb = __ldg(tau + 3 * s + 1), tc = __ldg(tau + 3 * s + 2);
        TC k1[DIM], k2[DIM], k3[DIM], k4[DIM], xi[DIM];
        ok = cart_velocity<DIM, TV, TC, FASTWRAP>(g, pa, ta, ci, w, k1);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) xi[a] = fma(TC(0.5) * hs[a], k1[a], w[a]);
        ok = cart_velocity<DIM, TV, TC, FASTWRAP>(g, pb, tb, ci, xi, k2);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) xi[a] = fma(TC(0.5) * hs[a], k2[a], w[a]);
        ok = cart_velocity<DIM, TV, TC, FASTWRAP>(g, pb, tb, ci, xi, k3);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) xi[a] = fma(hs[a], k3[a], w[a]);
        ok = cart_velocity<DIM, TV, TC, FASTWRAP>(g, pc, tc, ci, xi, k4);
        if (!ok) break;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            TC wn = fma(hs[a] * TC(1.0 / 6.0), (k1[a] + k4[a]) + TC(2) * (k2[a] + k3[a]), w[a]);
            TC fl = floor(wn);
            ci[a] += (int)fl;
            w[a] = wn - fl;
        }
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) { st.ci[a][i] = ci[a]; st.w[a][i] = w[a]; }
    if (!ok) { st.flag[i] = 1; st.steps[i] = first_step + s; }
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
    return g;
}

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

template <int DIM, typename TV, typename TC>
lcs_status cart_advect_impl(lcs_field *f, int64_t n, const void *seeds_, double t0, double h, int64_t N, void *flowmap_,
                            uint8_t *exit_flag, int32_t *exit_step, cudaStream_t st)
{
    const TC *seeds = (const TC *)seeds_;
    TC *flowmap = (TC *)flowmap_;
    std::vector<StepWindow> windows;
    std::vector<double> tau64;
    lcs_status rc = lcs_plan_windows(f, t0, h, N, windows, tau64);
    if (rc != LCS_OK) return rc;
    std::vector<TC> tau(tau64.size());
    for (size_t k = 0; k < tau.size(); ++k) tau[k] = (TC)tau64[k];

    // carve the tracer scratch
    size_t off = 0, o_ci[3], o_w[3], o_steps, o_flag, o_tau;
    for (int a = 0; a < DIM; ++a) { o_ci[a] = off; off = align_up(off + (size_t)n * 4); }
    for (int a = 0; a < DIM; ++a) { o_w[a] = off; off = align_up(off + (size_t)n * sizeof(TC)); }
    o_steps = off; off = align_up(off + (size_t)n * 4);
    o_flag = off; off = align_up(off + (size_t)n);
    o_tau = off; off = align_up(off + tau.size() * sizeof(TC));
    rc = lcs_scratch_reserve(f, off);
    if (rc != LCS_OK) return rc;
    char *base = (char *)f->scratch.buf;
    CartState<TC> S{};
    for (int a = 0; a < DIM; ++a) { S.ci[a] = (int32_t *)(base + o_ci[a]); S.w[a] = (TC *)(base + o_w[a]); }
    S.steps = (int32_t *)(base + o_steps);
    S.flag = (uint8_t *)(base + o_flag);
    TC *d_tau = (TC *)(base + o_tau);
    LCS_CUDA_OK(cudaMemcpyAsync(d_tau, tau.data(), tau.size() * sizeof(TC), cudaMemcpyHostToDevice, st));

    CartDev g = make_dev(f);
    const int block = f->opt_block ? (int)f->opt_block : 256;
    LCS_LAUNCH((cart_init_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, g, seeds, n, S);
    bool fast = true;
    for (int a = 0; a < DIM; ++a) fast = fast && g.periodic[a] && g.pow2[a];
    TC hs[3] = {TC(1), TC(1), TC(1)};
    for (int a = 0; a < DIM; ++a) hs[a] = (TC)(h * f->cart.inv[a]);
    const int dir = h > 0 ? 1 : -1;
    for (size_t wi = 0; wi < windows.size(); ++wi) {
        const StepWindow &w = windows[wi];
        const void *p[3];
        for (int k = 0; k < 3; ++k) {
            rc = lcs_field_require_pair(f, w.s[k], st, &p[k]);
            if (rc != LCS_OK) return rc;
        }
        // stream the snapshot the NEXT window will need while this one computes (side stream)
        lcs_field_prefetch(f, dir > 0 ? w.s[2] + 2 : w.s[2] - 1);
        using Rec = PairRec<DIM, TV>;
        WindowTimer timer(f, st);
        if (fast)
            LCS_LAUNCH((cart_window_kernel<DIM, TV, TC, true>), lcs_blocks(n, block), block, 0, st, g, (const Rec *)p[0], (const Rec *)p[1],
                       (const Rec *)p[2], d_tau + 3 * w.first, w.count, (int)w.first, n, S, hs[0], hs[1], hs[2]);
        else
            LCS_LAUNCH((cart_window_kernel<DIM, TV, TC, false>), lcs_blocks(n, block), block, 0, st, g, (const Rec *)p[0], (const Rec *)p[1],
                       (const Rec *)p[2], d_tau + 3 * w.first, w.count, (int)w.first, n, S, hs[0], hs[1], hs[2]);
        f->info_windows++;
    }
    LCS_LAUNCH((cart_final_kernel<DIM, TC>), lcs_blocks(n, 256), 256, 0, st, g, seeds, n, S, (int32_t)N, flowmap, exit_flag, exit_step);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

}  // namespace

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
        if (v64 && c64) return cart_advect_impl<2, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && c64) return cart_advect_impl<2, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && !c64) return cart_advect_impl<2, float, float>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    } else {
        if (v64 && c64) return cart_advect_impl<3, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && c64) return cart_advect_impl<3, double, double>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
        if (!v64 && !c64) return cart_advect_impl<3, float, float>(f, n, seeds, t0, h, N, flowmap, exit_flag, exit_step, st);
    }
    lcs_set_error("fp64 velocity with fp32 arithmetic is not supported (compute_dtype must be >= vel_dtype)");
    return LCS_ERR_INVALID_ARG;
}
