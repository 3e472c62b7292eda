// cg_ftle.cu -- fused finite-difference gradient (row a5), Cauchy-Green tensor and closed-form largest
// eigenvalue / FTLE (row a6) on the structured seed grid, for sm_100a.
//
// Paper: "standard central difference formula for the flow map gradient" on the seed grid;
// C = grad F^T grad F (Eq. 1.1); FTLE from the largest eigenvalue of C.
// The paper does not describe a GPU kernel for this stage (its GPU section covers the flow map only);
// here it is one HBM-streaming kernel: every flow-map element is read from DRAM once (the 2*dim stencil
// reads of neighbouring threads hit L1/L2), all arithmetic is fp64 (once per seed, far below the
// streaming time), outputs are written once.
#include <math.h>

#include "lcs_internal.cuh"

namespace {

struct CgGrid {
    int ng[3];
    int per[3];
    double inv_dx[3];     // 1/dx
    double period[3];
    double inv_2T;        // 1 / (2|T|)
};

__device__ __forceinline__ double eigmax_sym2(double c11, double c12, double c22)
{
    double hd = 0.5 * (c11 - c22);
    return 0.5 * (c11 + c22) + sqrt(hd * hd + c12 * c12);
}

// trigonometric closed form for the largest eigenvalue of a symmetric 3x3 matrix
__device__ __forceinline__ double eigmax_sym3(double c11, double c12, double c13, double c22, double c23, double c33)
{
    double q = (c11 + c22 + c33) / 3.0;
    double p1 = c12 * c12 + c13 * c13 + c23 * c23;
    double d1 = c11 - q, d2 = c22 - q, d3 = c33 - q;
    double p2 = d1 * d1 + d2 * d2 + d3 * d3 + 2.0 * p1;
    if (p2 == 0.0) return q;
    double p = sqrt(p2 / 6.0);
    double ip = 1.0 / p;
    double b11 = d1 * ip, b22 = d2 * ip, b33 = d3 * ip, b12 = c12 * ip, b13 = c13 * ip, b23 = c23 * ip;
    double det = b11 * (b22 * b33 - b23 * b23) - b12 * (b12 * b33 - b23 * b13) + b13 * (b12 * b23 - b22 * b13);
    double r = fmin(1.0, fmax(-1.0, 0.5 * det));
    return q + 2.0 * p * cos(acos(r) / 3.0);
}

// Single-precision outputs (T = float): C and the algebra of the eigenvalue stay in fp64, but the fp64 library routines
// (acos, cos, log: some hundred instructions each on the half-rate FP64 pipe, which made this HBM-streaming kernel FP64-bound
// at 20% of the HBM peak) are replaced: the trigonometric step runs in fp32 and its result is polished by one Newton step on the
// characteristic polynomial det(C - lambda I) in fp64 (taken only when it is a small correction: near a double root the
// determinant form is ill-conditioned and the kernel falls back to the fp64 closed form), and the logarithm of the float-rounded
// lambda_max is taken in fp32.  The result differs from the fp64 closed form by less than the rounding of the float output
// (tests: 2e-6 against the oracle).
// out of line: the rare fallback of eigmax_sym3_mixed must not cost the hot kernel registers (fp64 acos / cos are large)
__device__ __noinline__ double eigmax_sym3_rare(double c11, double c12, double c13, double c22, double c23, double c33)
{
    return eigmax_sym3(c11, c12, c13, c22, c23, c33);
}
__device__ __forceinline__ double eigmax_sym3_mixed(double c11, double c12, double c13, double c22, double c23, double c33)
{
    // estimate: the trigonometric closed form in fp32 (the largest eigenvalue of a symmetric matrix is well conditioned: the
    // estimate is within a few 1e-7 ||C||)
    const double qd = (c11 + c22 + c33) * (1.0 / 3.0);
    const float q = (float)qd;
    const float f12 = (float)c12, f13 = (float)c13, f23 = (float)c23;
    const float d1 = (float)(c11 - qd), d2 = (float)(c22 - qd), d3 = (float)(c33 - qd);
    const float p2 = d1 * d1 + d2 * d2 + d3 * d3 + 2.0f * (f12 * f12 + f13 * f13 + f23 * f23);
    if (!(p2 > 0.0f)) return qd;                               // multiple of the identity (or NaN, which propagates through qd)
    const float ip = rsqrtf(p2 * (1.0f / 6.0f));
    const float b11 = d1 * ip, b22 = d2 * ip, b33 = d3 * ip, b12 = f12 * ip, b13 = f13 * ip, b23 = f23 * ip;
    const float det = b11 * (b22 * b33 - b23 * b23) - b12 * (b12 * b33 - b23 * b13) + b13 * (b12 * b23 - b22 * b13);
    const float r = fminf(1.0f, fmaxf(-1.0f, 0.5f * det));
    const float pf = p2 * (1.0f / 6.0f) * ip;                  // sqrt(p2 / 6)
    double lam = qd + (double)(2.0f * pf * cosf(acosf(r) * (1.0f / 3.0f)));
    // one Newton step on det(C - lambda I) in fp64
    const double a11 = c11 - lam, a22 = c22 - lam, a33 = c33 - lam;
    const double m1 = a22 * a33 - c23 * c23, m2 = a11 * a33 - c13 * c13, m3 = a11 * a22 - c12 * c12;
    const double gv = a11 * m1 - c12 * (c12 * a33 - c23 * c13) + c13 * (c12 * c23 - a22 * c13);
    const double gd = -(m1 + m2 + m3);
    const double step = gv / gd;
    // The step measures the error e0 of the estimate: a few 1e-7 p far from a double root, about 1e-8 p / gap when the two largest
    // eigenvalues nearly coincide (the determinant form loses digits there), and the polished value is then off by e0^2 / gap.  Up to
    // e0 = 2e-5 p (relative gap above about 1e-3) that is below 5e-7 p, i.e. below the rounding of the float output; anything beyond
    // takes the fp64 closed form (rare: FTLE near zero).  NaN fails the comparison and takes it too (and stays NaN).
    if (fabs(step) <= 2e-5 * (double)pf) return lam - step;
    return eigmax_sym3_rare(c11, c12, c13, c22, c23, c33);
}
template <typename T> __device__ __forceinline__ double log_for(double lam)
{
    if constexpr (sizeof(T) == 4) {
        if (lam > 1e-30 && lam < 1e30) return (double)logf((float)lam);
    }
    return log(lam);
}

// EARLY (row f1, reading #29): the kernel runs at an evaluation point of lcs_advect_early_cg with the flags of
// that moment (0 alive, 1 left, 2 never started).  A seed is (re-)evaluated only if it is alive and none of its grid
// neighbours has left; neighbours that never started stay invalid neighbours (one-sided differences).  Seeds that are
// not evaluated keep the outputs of their previous evaluation; t_eff records the time of the last one.
template <int DIM, typename T, bool EARLY>
__global__ void __launch_bounds__(256) cg_ftle_kernel(const __grid_constant__ CgGrid g, const T *__restrict__ F,
                                                       const uint8_t *__restrict__ flag, T *__restrict__ cg,
                                                       T *__restrict__ ftle, uint8_t *__restrict__ status, int64_t n,
                                                       T *__restrict__ t_eff, double t_now)
{
    // launch geometry: x = position in the grid row, y / z = row and plane (no 64-bit division per seed: the index arithmetic of the
    // one-thread-per-linear-index version cost more issue slots than the whole eigenvalue)
    const int i0 = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    if (i0 >= g.ng[0]) return;
    const int64_t n0 = g.ng[0], n1 = g.ng[1];
    const int ijk[3] = {i0, (int)blockIdx.y, (int)blockIdx.z};
    const int64_t idx = i0 + n0 * (ijk[1] + n1 * (int64_t)ijk[2]);
    if (EARLY && flag[idx] != 0) return;
    const int64_t stride[3] = {1, n0, n0 * n1};
    constexpr int NCG = (DIM == 2) ? 3 : 6;
    uint8_t st = 0;
    if (flag && flag[idx] != 0) st = 1;
    double F0[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) F0[a] = (double)F[idx * DIM + a];
    double G[DIM][DIM];
#pragma unroll
    for (int b = 0; b < DIM; ++b) {
        int ip = ijk[b] + 1, im = ijk[b] - 1;
        double shp = 0.0, shm = 0.0;
        bool okp = true, okm = true;
        if (ip >= g.ng[b]) { if (g.per[b]) { ip -= g.ng[b]; shp = g.period[b]; } else okp = false; }
        if (im < 0) { if (g.per[b]) { im += g.ng[b]; shm = -g.period[b]; } else okm = false; }
        int64_t jp = idx + (int64_t)(ip - ijk[b]) * stride[b], jm = idx + (int64_t)(im - ijk[b]) * stride[b];
        if constexpr (EARLY) {
            if ((okp && flag[jp] == 1) || (okm && flag[jm] == 1)) return;
        }
        if (okp && flag && flag[jp] != 0) okp = false;
        if (okm && flag && flag[jm] != 0) okm = false;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            double Fp = okp ? (double)F[jp * DIM + a] + (a == b ? shp : 0.0) : 0.0;
            double Fm = okm ? (double)F[jm * DIM + a] + (a == b ? shm : 0.0) : 0.0;
            double v = 0.0;
            if (okp && okm) v = (Fp - Fm) * (0.5 * g.inv_dx[b]);
            else if (okp) v = (Fp - F0[a]) * g.inv_dx[b];
            else if (okm) v = (F0[a] - Fm) * g.inv_dx[b];
            G[a][b] = v;
        }
        // status bits accumulate axis by axis until the seed becomes undefined (as the oracle's rule O5 does)
        if (!(st & 1)) {
            if (!okp && !okm) st |= 1;
            else if (!(okp && okm)) st |= 2;
        }
    }
    double C[NCG], lam;
    if (st & 1) {
#pragma unroll
        for (int i = 0; i < NCG; ++i) C[i] = nan("");
        lam = nan("");
    } else if constexpr (DIM == 2) {
        C[0] = G[0][0] * G[0][0] + G[1][0] * G[1][0];
        C[1] = G[0][0] * G[0][1] + G[1][0] * G[1][1];
        C[2] = G[0][1] * G[0][1] + G[1][1] * G[1][1];
        lam = eigmax_sym2(C[0], C[1], C[2]);
    } else {
        int m = 0;
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int c = b; c < 3; ++c) C[m++] = G[0][b] * G[0][c] + G[1][b] * G[1][c] + G[2][b] * G[2][c];
        lam = sizeof(T) == 4 ? eigmax_sym3_mixed(C[0], C[1], C[2], C[3], C[4], C[5]) : eigmax_sym3(C[0], C[1], C[2], C[3], C[4], C[5]);
    }
    if (cg) {
        if constexpr (sizeof(T) == 4 && NCG == 6) {
            // 24 bytes per seed, 8-byte aligned: three 64-bit stores instead of six 32-bit ones
            float2 *o = reinterpret_cast<float2 *>(cg + idx * NCG);
            o[0] = make_float2((float)C[0], (float)C[1]);
            o[1] = make_float2((float)C[2], (float)C[3]);
            o[2] = make_float2((float)C[4], (float)C[5]);
        } else {
#pragma unroll
            for (int i = 0; i < NCG; ++i) cg[idx * NCG + i] = (T)C[i];
        }
    }
    ftle[idx] = (st & 1) ? (T)nan("") : (T)(log_for<T>(lam) * g.inv_2T);
    if (status) status[idx] = st;
    if constexpr (EARLY) t_eff[idx] = (T)t_now;
}

// The hot instantiation (3D, float, plain evaluation: configs 3-5) written for issue slots: the generic kernel above spends 710
// instructions per seed, a fifth of them on 64-bit index arithmetic and another tenth on branches, and runs at 20% of the HBM
// peak although it moves 42 bytes per seed (ncu: issue slots 72%, DRAM 16%).  Here the neighbour offsets are 32-bit, validity is
// carried in predicates (loads are issued for every in-grid neighbour whatever its flag), the selection between central and
// one-sided differences happens on the float operands before ONE widening subtraction per entry, and C leaves in three 64-bit
// stores.  Same rule (reading #12) and the same fp64 arithmetic for the differences, C and the eigenvalue algebra.
// Requires 3 n < 2^31 (32-bit element offsets).
template <bool PER_ALL> __global__ void __launch_bounds__(256, 6) cg_ftle3f_kernel(const __grid_constant__ CgGrid g, const float *__restrict__ F, const uint8_t *__restrict__ flag,
                                                         float *__restrict__ cg, float *__restrict__ ftle, uint8_t *__restrict__ status)
{
    const int i0 = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    if (i0 >= g.ng[0]) return;
    const unsigned lanes = __activemask();
    const int n0 = g.ng[0], n1 = g.ng[1], n2 = g.ng[2];
    const int ijk[3] = {i0, (int)blockIdx.y, (int)blockIdx.z};
    const int nn[3] = {n0, n1, n2};
    const int stride[3] = {1, n0, n0 * n1};
    const int idx = i0 + n0 * (ijk[1] + n1 * ijk[2]);
    // in-grid neighbours (by wrap on a periodic axis), their flags
    bool atp[3], atm[3], okp[3], okm[3];
    int jp[3], jm[3];
    bool all_ok = !(flag && flag[idx] != 0);
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        atp[b] = ijk[b] + 1 >= nn[b];
        atm[b] = ijk[b] == 0;
        okp[b] = PER_ALL || !atp[b] || g.per[b];               // PER_ALL: every axis wraps, every neighbour is in the grid
        okm[b] = PER_ALL || !atm[b] || g.per[b];
        jp[b] = okp[b] ? idx + (atp[b] ? 1 - nn[b] : 1) * stride[b] : idx;        // a valid address in every case
        jm[b] = okm[b] ? idx + (atm[b] ? nn[b] - 1 : -1) * stride[b] : idx;
        if (flag) { okp[b] = okp[b] && flag[jp[b]] == 0; okm[b] = okm[b] && flag[jm[b]] == 0; }
        all_ok = all_ok && okp[b] && okm[b];
    }
    double G[3][3];
    unsigned st = 0;
    if (__all_sync(lanes, all_ok)) {
        // every seed of the warp has its full stencil (the whole of configs 3 and 5): central differences without selects
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const float *Pp = F + 3 * jp[b], *Pm = F + 3 * jm[b];
            const double shift = (atp[b] ? g.period[b] : 0.0) + (atm[b] ? g.period[b] : 0.0);
            const double scale = 0.5 * g.inv_dx[b];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                double d = (double)Pp[a] - (double)Pm[a];
                if (a == b) d += shift;
                G[a][b] = d * scale;
            }
        }
    } else {
        const float *Fc = F + 3 * idx;
        const float F0[3] = {Fc[0], Fc[1], Fc[2]};
        st = (flag && flag[idx] != 0) ? 1u : 0u;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const float *Pp = F + 3 * jp[b], *Pm = F + 3 * jm[b];
            const float fp[3] = {Pp[0], Pp[1], Pp[2]}, fm[3] = {Pm[0], Pm[1], Pm[2]};
            const double shift = ((okp[b] && atp[b]) ? g.period[b] : 0.0) + ((okm[b] && atm[b]) ? g.period[b] : 0.0);
            const double scale = (okp[b] && okm[b]) ? 0.5 * g.inv_dx[b] : ((okp[b] || okm[b]) ? g.inv_dx[b] : 0.0);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float hi = okp[b] ? fp[a] : F0[a], lo = okm[b] ? fm[a] : F0[a];
                double d = (double)hi - (double)lo;
                if (a == b) d += shift;
                G[a][b] = d * scale;
            }
            if (!(st & 1u)) {
                if (!okp[b] && !okm[b]) st |= 1u;
                else if (!(okp[b] && okm[b])) st |= 2u;
            }
        }
    }
    float c[6], ft;
    if (st & 1u) {
        const float q = __int_as_float(0x7fc00000);
#pragma unroll
        for (int i = 0; i < 6; ++i) c[i] = q;
        ft = q;
    } else {
        double C[6];
        int m = 0;
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int k = b; k < 3; ++k) C[m++] = G[0][b] * G[0][k] + G[1][b] * G[1][k] + G[2][b] * G[2][k];
        const double lam = eigmax_sym3_mixed(C[0], C[1], C[2], C[3], C[4], C[5]);
        ft = (float)(log_for<float>(lam) * g.inv_2T);
#pragma unroll
        for (int i = 0; i < 6; ++i) c[i] = (float)C[i];
    }
    if (cg) {
        float2 *o = reinterpret_cast<float2 *>(cg + 6 * (int64_t)idx);
        o[0] = make_float2(c[0], c[1]);
        o[1] = make_float2(c[2], c[3]);
        o[2] = make_float2(c[4], c[5]);
    }
    ftle[idx] = ft;
    if (status) status[idx] = (uint8_t)st;
}

// outputs of seeds that are never evaluated: NaN, t_eff = 0, status bit 0
template <typename T>
__global__ void __launch_bounds__(256) early_init_kernel(T *__restrict__ cg, int ncg, T *__restrict__ ftle, T *__restrict__ t_eff,
                                                          uint8_t *__restrict__ status, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const T q = (T)nan("");
    if (cg) for (int k = 0; k < ncg; ++k) cg[i * ncg + k] = q;
    ftle[i] = q;
    t_eff[i] = T(0);
    if (status) status[i] = 1;
}

// ---------------------------------------------------------------------------------------------
// Row f3: gradient from auxiliary points ("auxiliary points can be placed around each seed point",
// PAPER.md:67 "used for the computation of the flow map gradient").  Faux: [n][2 DIM][DIM], entry 2b / 2b+1 = final
// position of the tracer released at x0 +/- delta_b e_b; always central; any flagged auxiliary tracer => NaN, status 1
// (reading #28).  HBM streaming: 2 DIM^2 elements in per seed, read once, fully coalesced across the warp.
template <int DIM, typename T>
__global__ void __launch_bounds__(256) cg_ftle_aux_kernel(const T *__restrict__ Faux, const uint8_t *__restrict__ flag_aux,
                                                           double i2d0, double i2d1, double i2d2, double inv_2T, T *__restrict__ cg,
                                                           T *__restrict__ ftle, uint8_t *__restrict__ status, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    constexpr int NCG = (DIM == 2) ? 3 : 6;
    const double i2d[3] = {i2d0, i2d1, i2d2};
    uint8_t st = 0;
    if (flag_aux) {
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) st |= flag_aux[i * 2 * DIM + k] != 0 ? 1 : 0;
    }
    double G[DIM][DIM];
    const T *f = Faux + i * (2 * DIM * DIM);
#pragma unroll
    for (int b = 0; b < DIM; ++b)
#pragma unroll
        for (int a = 0; a < DIM; ++a) G[a][b] = ((double)f[(2 * b) * DIM + a] - (double)f[(2 * b + 1) * DIM + a]) * i2d[b];
    double C[NCG], lam;
    if (st) {
#pragma unroll
        for (int k = 0; k < NCG; ++k) C[k] = nan("");
        lam = nan("");
    } else if constexpr (DIM == 2) {
        C[0] = G[0][0] * G[0][0] + G[1][0] * G[1][0];
        C[1] = G[0][0] * G[0][1] + G[1][0] * G[1][1];
        C[2] = G[0][1] * G[0][1] + G[1][1] * G[1][1];
        lam = eigmax_sym2(C[0], C[1], C[2]);
    } else {
        int m = 0;
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int c = b; c < 3; ++c) C[m++] = G[0][b] * G[0][c] + G[1][b] * G[1][c] + G[2][b] * G[2][c];
        lam = sizeof(T) == 4 ? eigmax_sym3_mixed(C[0], C[1], C[2], C[3], C[4], C[5]) : eigmax_sym3(C[0], C[1], C[2], C[3], C[4], C[5]);
    }
    if (cg) {
#pragma unroll
        for (int k = 0; k < NCG; ++k) cg[i * NCG + k] = (T)C[k];
    }
    ftle[i] = st ? (T)nan("") : (T)(log_for<T>(lam) * inv_2T);
    if (status) status[i] = st;
}

// ---------------------------------------------------------------------------------------------
// Row f4 (first part): Gaussian smoothing of the FTLE field before ridge extraction, reading #30.
// One normalised 1D convolution per axis (radius ceil(3 sigma) <= 64, weights in shared memory), NaN centres kept, NaN and
// out-of-grid neighbours skipped with renormalisation, fp64 accumulation.  HBM streaming: one read + one write per pass;
// the 2R+1 taps of neighbouring threads hit L1 / L2.
template <typename T>
__global__ void __launch_bounds__(256) smooth_axis_kernel(const T *__restrict__ in, T *__restrict__ out, int64_t total, int64_t stride,
                                                           int64_t len, int periodic, int R, double inv_2s2)
{
    __shared__ double w[65];
    for (int k = threadIdx.x; k <= R; k += blockDim.x) w[k] = exp(-(double)(k * k) * inv_2s2);
    __syncthreads();
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const T centre = in[idx];
    if (!isfinite((double)centre)) { out[idx] = centre; return; }
    const int64_t i = (idx / stride) % len;
    double num = 0.0, den = 0.0;
    for (int k = -R; k <= R; ++k) {
        int64_t j = i + k;
        if (periodic) { j %= len; if (j < 0) j += len; }
        else if (j < 0 || j >= len) continue;
        const double v = (double)in[idx + (j - i) * stride];
        if (!isfinite(v)) continue;
        const double wk = w[k < 0 ? -k : k];
        num = fma(wk, v, num);
        den += wk;
    }
    out[idx] = (T)(num / den);
}

// ---------------------------------------------------------------------------------------------
// Row f2: all eigenvalues and eigenvectors of C ("eigenvalues and eigenvectors"; the
// eigenvector fields are what hyperbolic-LCS criteria need).  One thread per seed, cyclic Jacobi in fp64 registers
// (reading #27): the closed forms are ill-conditioned for the small eigenvalues.  Streams 12-24 B in and
// 24-48 B out per seed (fp32); the arithmetic is FP64-pipe bound.
template <int D> __device__ __forceinline__ void jacobi_rotate(double (&a)[D][D], double (&v)[D][D], int p, int q)
{
    const double apq = a[p][q];
    if (apq == 0.0) return;
    const double theta = (a[q][q] - a[p][p]) / (2.0 * apq);
    double t = copysign(1.0, theta) / (fabs(theta) + sqrt(fma(theta, theta, 1.0)));
    if (!isfinite(theta)) t = 0.0;
    const double c = rsqrt(fma(t, t, 1.0)), s = t * c;
    a[p][p] -= t * apq;
    a[q][q] += t * apq;
    a[p][q] = a[q][p] = 0.0;
#pragma unroll
    for (int r = 0; r < D; ++r) {
        if (r != p && r != q) {
            const double arp = a[r][p], arq = a[r][q];
            a[r][p] = a[p][r] = c * arp - s * arq;
            a[r][q] = a[q][r] = s * arp + c * arq;
        }
        const double vrp = v[r][p], vrq = v[r][q];
        v[r][p] = c * vrp - s * vrq;
        v[r][q] = s * vrp + c * vrq;
    }
}

// ---------------------------------------------------------------------------------------------
// Row f4 (third part): ridge indicator of the (smoothed) FTLE field ("C-ridge extraction"; DESIGN.md reading
// #32: second-derivative ridge).  Per seed: gradient and Hessian by central differences on the 3^d stencil, smallest
// Hessian eigenvalue kappa and its eigenvector n by Jacobi in fp64, d = g . n, mask = kappa < -kappa_min && s >= s_min &&
// |d| <= |kappa| delta / 2.  Streams the field once (stencil taps hit L1/L2); FP64-pipe bound like the eigen kernels.
struct RidgeGrid {
    int ng[3], per[3];
    double dx[3];
    double kappa_min, s_min, delta;
};

template <int D, typename T>
__global__ void __launch_bounds__(128) ridge_kernel(const __grid_constant__ RidgeGrid g, const T *__restrict__ field, T *__restrict__ kappa,
                                                     T *__restrict__ dgn, uint8_t *__restrict__ mask, int64_t total)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int64_t n0 = g.ng[0], n1 = g.ng[1];
    const int64_t ijk[3] = {idx % n0, (idx / n0) % n1, idx / (n0 * n1)};
    const int64_t stride[3] = {1, n0, n0 * n1};
    int64_t off[D][3];
    bool ok = true;
#pragma unroll
    for (int a = 0; a < D; ++a)
#pragma unroll
        for (int k = -1; k <= 1; ++k) {
            int64_t j = ijk[a] + k;
            if (j < 0 || j >= g.ng[a]) { if (g.per[a]) j = (j + g.ng[a]) % g.ng[a]; else ok = false; }
            off[a][k + 1] = (j - ijk[a]) * stride[a];
        }
    double gr[D], H[D][D], v[D][D];
    const double s0 = ok ? (double)field[idx] : 0.0;
    ok = ok && isfinite(s0);
    if (ok) {
#pragma unroll
        for (int a = 0; a < D; ++a) {
            const double sp = (double)field[idx + off[a][2]], sm = (double)field[idx + off[a][0]];
            ok = ok && isfinite(sp) && isfinite(sm);
            gr[a] = (sp - sm) / (2.0 * g.dx[a]);
            H[a][a] = (sp - 2.0 * s0 + sm) / (g.dx[a] * g.dx[a]);
#pragma unroll
            for (int b = a + 1; b < D; ++b) {
                const double pp = (double)field[idx + off[a][2] + off[b][2]], pm = (double)field[idx + off[a][2] + off[b][0]];
                const double mp = (double)field[idx + off[a][0] + off[b][2]], mm = (double)field[idx + off[a][0] + off[b][0]];
                ok = ok && isfinite(pp) && isfinite(pm) && isfinite(mp) && isfinite(mm);
                H[a][b] = H[b][a] = (pp - pm - mp + mm) / (4.0 * g.dx[a] * g.dx[b]);
            }
        }
    }
    if (!ok) {
        kappa[idx] = (T)nan(""); dgn[idx] = (T)nan(""); mask[idx] = 0;
        return;
    }
#pragma unroll
    for (int r = 0; r < D; ++r)
#pragma unroll
        for (int k = 0; k < D; ++k) v[r][k] = r == k ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 50; ++sweep) {
        double offd = fabs(H[0][1]);
        if constexpr (D == 3) offd += fabs(H[0][2]) + fabs(H[1][2]);
        if (offd == 0.0) break;
        jacobi_rotate<D>(H, v, 0, 1);
        if constexpr (D == 3) { jacobi_rotate<D>(H, v, 0, 2); jacobi_rotate<D>(H, v, 1, 2); }
    }
    double kap = H[0][0], nv[D];
#pragma unroll
    for (int r = 0; r < D; ++r) nv[r] = v[r][0];
#pragma unroll
    for (int k = 1; k < D; ++k)
        if (H[k][k] < kap) {
            kap = H[k][k];
#pragma unroll
            for (int r = 0; r < D; ++r) nv[r] = v[r][k];
        }
    double big = nv[0];
#pragma unroll
    for (int r = 1; r < D; ++r)
        if (fabs(nv[r]) > fabs(big)) big = nv[r];
    const double sg = big < 0.0 ? -1.0 : 1.0;
    double d = 0.0;
#pragma unroll
    for (int r = 0; r < D; ++r) d += gr[r] * (sg * nv[r]);
    kappa[idx] = (T)kap;
    dgn[idx] = (T)d;
    mask[idx] = (kap < -g.kappa_min && s0 >= g.s_min && fabs(d) <= fabs(kap) * g.delta * 0.5) ? 1 : 0;
}

template <int D, typename T>
__global__ void __launch_bounds__(128) cg_eigen_kernel(const T *__restrict__ cg, T *__restrict__ evals, T *__restrict__ evecs, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    constexpr int NCG = D == 2 ? 3 : 6;
    double c[NCG];
    bool finite = true;
#pragma unroll
    for (int k = 0; k < NCG; ++k) { c[k] = (double)cg[i * NCG + k]; finite = finite && isfinite(c[k]); }
    if (!finite) {
        const T q = (T)nan("");
#pragma unroll
        for (int k = 0; k < D; ++k) evals[i * D + k] = q;
#pragma unroll
        for (int k = 0; k < D * D; ++k) evecs[i * D * D + k] = q;
        return;
    }
    double a[D][D], v[D][D];
    if constexpr (D == 2) { a[0][0] = c[0]; a[0][1] = a[1][0] = c[1]; a[1][1] = c[2]; }
    else { a[0][0] = c[0]; a[0][1] = a[1][0] = c[1]; a[0][2] = a[2][0] = c[2]; a[1][1] = c[3]; a[1][2] = a[2][1] = c[4]; a[2][2] = c[5]; }
#pragma unroll
    for (int r = 0; r < D; ++r)
#pragma unroll
        for (int k = 0; k < D; ++k) v[r][k] = r == k ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 50; ++sweep) {
        double off = fabs(a[0][1]);
        if constexpr (D == 3) off += fabs(a[0][2]) + fabs(a[1][2]);
        if (off == 0.0) break;
        jacobi_rotate<D>(a, v, 0, 1);
        if constexpr (D == 3) { jacobi_rotate<D>(a, v, 0, 2); jacobi_rotate<D>(a, v, 1, 2); }
    }
    // ascending order by a 2- or 3-element sorting network on (eigenvalue, column)
    double ev[D], col[D][D];
#pragma unroll
    for (int k = 0; k < D; ++k) {
        ev[k] = a[k][k];
#pragma unroll
        for (int r = 0; r < D; ++r) col[k][r] = v[r][k];
    }
    auto cswap = [&](int x, int y) {
        if (ev[y] < ev[x]) {
            double t = ev[x]; ev[x] = ev[y]; ev[y] = t;
#pragma unroll
            for (int r = 0; r < D; ++r) { double u = col[x][r]; col[x][r] = col[y][r]; col[y][r] = u; }
        }
    };
    cswap(0, 1);
    if constexpr (D == 3) { cswap(1, 2); cswap(0, 1); }
#pragma unroll
    for (int k = 0; k < D; ++k) {
        double big = col[k][0];
#pragma unroll
        for (int r = 1; r < D; ++r)
            if (fabs(col[k][r]) > fabs(big)) big = col[k][r];
        const double sg = big < 0.0 ? -1.0 : 1.0;
        evals[i * D + k] = (T)ev[k];
#pragma unroll
        for (int r = 0; r < D; ++r) evecs[(i * D + k) * D + r] = (T)(sg * col[k][r]);
    }
}

}  // namespace

extern "C" lcs_status lcs_cg_ftle(int32_t dim, int32_t dtype, const int32_t ng[3], const double seed_spacing[3],
                                  const int32_t seed_periodic[3], const double period[3], const void *flowmap,
                                  const uint8_t *exit_flag, double T, void *cg, void *ftle, uint8_t *status, void *cuda_stream)
{
    if ((dim != 2 && dim != 3) || !ng || !seed_spacing || !flowmap || !ftle) { lcs_set_error("null argument or bad dim"); return LCS_ERR_INVALID_ARG; }
    if (dtype != LCS_F32 && dtype != LCS_F64) { lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG; }
    if (!(T != 0.0) || !isfinite(T)) { lcs_set_error("T must be finite and non-zero"); return LCS_ERR_INVALID_ARG; }
    CgGrid g;
    int64_t n = 1;
    for (int a = 0; a < 3; ++a) {
        g.ng[a] = a < dim ? ng[a] : 1;
        g.per[a] = (a < dim && seed_periodic) ? (seed_periodic[a] != 0) : 0;
        g.period[a] = (a < dim && period) ? period[a] : 0.0;
        if (a < dim && (ng[a] < 1 || !(seed_spacing[a] > 0))) { lcs_set_error("bad seed grid on axis %d", a); return LCS_ERR_INVALID_ARG; }
        g.inv_dx[a] = a < dim ? 1.0 / seed_spacing[a] : 1.0;
        n *= g.ng[a];
    }
    g.inv_2T = 1.0 / (2.0 * fabs(T));
    if (n == 0) return LCS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // one thread per seed of a grid row; rows and planes on the y / z axes of the launch grid
    if (g.ng[1] > 65535 || g.ng[2] > 65535) { lcs_set_error("seed grid too large on axis 1 or 2 (max 65535)"); return LCS_ERR_INVALID_ARG; }
    const unsigned bx = (unsigned)(g.ng[0] >= 256 ? 256 : ((g.ng[0] + 31) / 32) * 32);
    const dim3 block3(bx, 1, 1), grid3((unsigned)((g.ng[0] + bx - 1) / bx), (unsigned)g.ng[1], (unsigned)g.ng[2]);
    if (dim == 2 && dtype == LCS_F64) LCS_LAUNCH((cg_ftle_kernel<2, double, false>), grid3, block3, 0, st, g, (const double *)flowmap, exit_flag, (double *)cg, (double *)ftle, status, n, (double *)nullptr, 0.0);
    else if (dim == 2) LCS_LAUNCH((cg_ftle_kernel<2, float, false>), grid3, block3, 0, st, g, (const float *)flowmap, exit_flag, (float *)cg, (float *)ftle, status, n, (float *)nullptr, 0.0);
    else if (dtype == LCS_F64) LCS_LAUNCH((cg_ftle_kernel<3, double, false>), grid3, block3, 0, st, g, (const double *)flowmap, exit_flag, (double *)cg, (double *)ftle, status, n, (double *)nullptr, 0.0);
    else if (3 * n < (1LL << 31) && g.per[0] && g.per[1] && g.per[2])
        LCS_LAUNCH(cg_ftle3f_kernel<true>, grid3, block3, 0, st, g, (const float *)flowmap, exit_flag, (float *)cg, (float *)ftle, status);
    else if (3 * n < (1LL << 31)) LCS_LAUNCH(cg_ftle3f_kernel<false>, grid3, block3, 0, st, g, (const float *)flowmap, exit_flag, (float *)cg, (float *)ftle, status);
    else LCS_LAUNCH((cg_ftle_kernel<3, float, false>), grid3, block3, 0, st, g, (const float *)flowmap, exit_flag, (float *)cg, (float *)ftle, status, n, (float *)nullptr, 0.0);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

extern "C" lcs_status lcs_cg_eigen(int32_t dim, int32_t dtype, int64_t n, const void *cg, void *evals, void *evecs, void *cuda_stream)
{
    if ((dim != 2 && dim != 3) || n < 0 || (n > 0 && (!cg || !evals || !evecs))) { lcs_set_error("null argument or bad dim"); return LCS_ERR_INVALID_ARG; }
    if (dtype != LCS_F32 && dtype != LCS_F64) { lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG; }
    if (n == 0) return LCS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = lcs_blocks(n, 128);
    if (dim == 2 && dtype == LCS_F64) LCS_LAUNCH((cg_eigen_kernel<2, double>), grid, 128, 0, st, (const double *)cg, (double *)evals, (double *)evecs, n);
    else if (dim == 2) LCS_LAUNCH((cg_eigen_kernel<2, float>), grid, 128, 0, st, (const float *)cg, (float *)evals, (float *)evecs, n);
    else if (dtype == LCS_F64) LCS_LAUNCH((cg_eigen_kernel<3, double>), grid, 128, 0, st, (const double *)cg, (double *)evals, (double *)evecs, n);
    else LCS_LAUNCH((cg_eigen_kernel<3, float>), grid, 128, 0, st, (const float *)cg, (float *)evals, (float *)evecs, n);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

extern "C" lcs_status lcs_cg_ftle_aux(int32_t dim, int32_t dtype, int64_t n, const double aux_delta[3], const void *flowmap_aux,
                                      const uint8_t *exit_flag_aux, double T, void *cg, void *ftle, uint8_t *status, void *cuda_stream)
{
    if ((dim != 2 && dim != 3) || n < 0 || !aux_delta || (n > 0 && (!flowmap_aux || !ftle))) { lcs_set_error("null argument or bad dim"); return LCS_ERR_INVALID_ARG; }
    if (dtype != LCS_F32 && dtype != LCS_F64) { lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG; }
    if (!(T != 0.0) || !isfinite(T)) { lcs_set_error("T must be finite and non-zero"); return LCS_ERR_INVALID_ARG; }
    double i2d[3] = {1.0, 1.0, 1.0};
    for (int a = 0; a < dim; ++a) {
        if (!(aux_delta[a] > 0.0) || !isfinite(aux_delta[a])) { lcs_set_error("aux_delta[%d] must be positive", a); return LCS_ERR_INVALID_ARG; }
        i2d[a] = 1.0 / (2.0 * aux_delta[a]);
    }
    if (n == 0) return LCS_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = lcs_blocks(n, 256);
    const double inv_2T = 1.0 / (2.0 * fabs(T));
    if (dim == 2 && dtype == LCS_F64) LCS_LAUNCH((cg_ftle_aux_kernel<2, double>), grid, 256, 0, st, (const double *)flowmap_aux, exit_flag_aux, i2d[0], i2d[1], i2d[2], inv_2T, (double *)cg, (double *)ftle, status, n);
    else if (dim == 2) LCS_LAUNCH((cg_ftle_aux_kernel<2, float>), grid, 256, 0, st, (const float *)flowmap_aux, exit_flag_aux, i2d[0], i2d[1], i2d[2], inv_2T, (float *)cg, (float *)ftle, status, n);
    else if (dtype == LCS_F64) LCS_LAUNCH((cg_ftle_aux_kernel<3, double>), grid, 256, 0, st, (const double *)flowmap_aux, exit_flag_aux, i2d[0], i2d[1], i2d[2], inv_2T, (double *)cg, (double *)ftle, status, n);
    else LCS_LAUNCH((cg_ftle_aux_kernel<3, float>), grid, 256, 0, st, (const float *)flowmap_aux, exit_flag_aux, i2d[0], i2d[1], i2d[2], inv_2T, (float *)cg, (float *)ftle, status, n);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
// Row f1: early evaluation of C when a stencil member leaves the domain
lcs_status lcs_early_cg_eval(lcs_field *f, int64_t m, cudaStream_t st)
{
    const EarlyCg &e = f->early;
    CgGrid g;
    int64_t n = 1;
    for (int a = 0; a < 3; ++a) {
        g.ng[a] = e.ng[a]; g.per[a] = e.per[a]; g.period[a] = e.period[a]; g.inv_dx[a] = 1.0 / e.dx[a];
        n *= e.ng[a];
    }
    const double t_now = (double)m * e.h;
    g.inv_2T = 1.0 / (2.0 * fabs(t_now));
    // one thread per seed of a grid row; rows and planes on the y / z axes of the launch grid
    if (g.ng[1] > 65535 || g.ng[2] > 65535) { lcs_set_error("seed grid too large on axis 1 or 2 (max 65535)"); return LCS_ERR_INVALID_ARG; }
    const unsigned bx = (unsigned)(g.ng[0] >= 256 ? 256 : ((g.ng[0] + 31) / 32) * 32);
    const dim3 block3(bx, 1, 1), grid3((unsigned)((g.ng[0] + bx - 1) / bx), (unsigned)g.ng[1], (unsigned)g.ng[2]);
    const bool f64 = f->compute_dtype == LCS_F64;
    if (f->dim == 2 && f64) LCS_LAUNCH((cg_ftle_kernel<2, double, true>), grid3, block3, 0, st, g, (const double *)e.flowmap, e.flag, (double *)e.cg, (double *)e.ftle, e.status, n, (double *)e.t_eff, t_now);
    else if (f->dim == 2) LCS_LAUNCH((cg_ftle_kernel<2, float, true>), grid3, block3, 0, st, g, (const float *)e.flowmap, e.flag, (float *)e.cg, (float *)e.ftle, e.status, n, (float *)e.t_eff, t_now);
    else if (f64) LCS_LAUNCH((cg_ftle_kernel<3, double, true>), grid3, block3, 0, st, g, (const double *)e.flowmap, e.flag, (double *)e.cg, (double *)e.ftle, e.status, n, (double *)e.t_eff, t_now);
    else LCS_LAUNCH((cg_ftle_kernel<3, float, true>), grid3, block3, 0, st, g, (const float *)e.flowmap, e.flag, (float *)e.cg, (float *)e.ftle, e.status, n, (float *)e.t_eff, t_now);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

extern "C" lcs_status lcs_advect_early_cg(lcs_field *f, const int32_t ng[3], const double seed_spacing[3], const int32_t seed_periodic[3],
                                          const double period[3], const void *seeds, double t0, double tf, double h, int32_t every,
                                          void *flowmap, uint8_t *exit_flag, int32_t *exit_step, void *cg, void *ftle, void *t_eff,
                                          uint8_t *status, void *cuda_stream)
{
    if (!f || !ng || !seed_spacing || !seeds || !flowmap || !exit_flag || !ftle || !t_eff) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    if (every < 1) { lcs_set_error("every must be >= 1"); return LCS_ERR_INVALID_ARG; }
    if (flowmap == seeds) { lcs_set_error("flowmap must not alias seeds (it is rewritten at every evaluation point)"); return LCS_ERR_INVALID_ARG; }
    EarlyCg e;
    int64_t n = 1;
    for (int a = 0; a < 3; ++a) {
        e.ng[a] = a < f->dim ? ng[a] : 1;
        e.per[a] = (a < f->dim && seed_periodic) ? (seed_periodic[a] != 0) : 0;
        e.period[a] = (a < f->dim && period) ? period[a] : 0.0;
        e.dx[a] = a < f->dim ? seed_spacing[a] : 1.0;
        if (a < f->dim && (ng[a] < 1 || !(seed_spacing[a] > 0))) { lcs_set_error("bad seed grid on axis %d", a); return LCS_ERR_INVALID_ARG; }
        n *= e.ng[a];
    }
    e.on = true; e.every = every; e.h = h;
    e.flowmap = flowmap; e.flag = exit_flag; e.cg = cg; e.ftle = ftle; e.t_eff = t_eff; e.status = status;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int ncg = f->dim == 2 ? 3 : 6;
    if (f->compute_dtype == LCS_F64) LCS_LAUNCH((early_init_kernel<double>), lcs_blocks(n, 256), 256, 0, st, (double *)cg, ncg, (double *)ftle, (double *)t_eff, status, n);
    else LCS_LAUNCH((early_init_kernel<float>), lcs_blocks(n, 256), 256, 0, st, (float *)cg, ncg, (float *)ftle, (float *)t_eff, status, n);
    f->early = e;
    lcs_status rc = lcs_advect(f, n, seeds, t0, tf, h, flowmap, exit_flag, exit_step, cuda_stream);
    f->early = EarlyCg();
    return rc;
}

extern "C" lcs_status lcs_smooth_gaussian(int32_t dim, int32_t dtype, const int32_t ng[3], const int32_t seed_periodic[3], double sigma,
                                          const void *field, void *out, void *work, void *cuda_stream)
{
    if ((dim != 2 && dim != 3) || !ng || !field || !out || !work) { lcs_set_error("null argument or bad dim"); return LCS_ERR_INVALID_ARG; }
    if (dtype != LCS_F32 && dtype != LCS_F64) { lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG; }
    if (!(sigma > 0.0) || ceil(3.0 * sigma) > 64.0) { lcs_set_error("sigma must be in (0, 21.33] seed-grid cells"); return LCS_ERR_INVALID_ARG; }
    if (out == field || work == field || work == out) { lcs_set_error("field, out and work must be distinct buffers"); return LCS_ERR_INVALID_ARG; }
    int64_t n[3] = {1, 1, 1}, total = 1;
    for (int a = 0; a < dim; ++a) { if (ng[a] < 1) { lcs_set_error("bad seed grid"); return LCS_ERR_INVALID_ARG; } n[a] = ng[a]; total *= n[a]; }
    const int64_t stride[3] = {1, n[0], n[0] * n[1]};
    const int R = (int)ceil(3.0 * sigma);
    const double inv_2s2 = 1.0 / (2.0 * sigma * sigma);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // dim passes ending in `out`: 2D: field -> work -> out; 3D: field -> out -> work -> out
    const void *src = field;
    for (int a = 0; a < dim; ++a) {
        void *dst = ((dim - a) % 2 == 1) ? out : work;
        const int per = seed_periodic ? (seed_periodic[a] != 0) : 0;
        if (dtype == LCS_F64) LCS_LAUNCH((smooth_axis_kernel<double>), lcs_blocks(total, 256), 256, 0, st, (const double *)src, (double *)dst, total, stride[a], n[a], per, R, inv_2s2);
        else LCS_LAUNCH((smooth_axis_kernel<float>), lcs_blocks(total, 256), 256, 0, st, (const float *)src, (float *)dst, total, stride[a], n[a], per, R, inv_2s2);
        src = dst;
    }
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

// ---------------------------------------------------------------------------------------------
// lcs_smooth_gaussian without a caller-supplied work buffer and without any allocation: the intermediate field of the axis passes
// lives in a file-scope device array.  For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses
// that forbid it).  Every GPU that loads the library holds the array (16 MiB) until the process exits.
constexpr size_t kSmoothScratchBytes = (size_t)16 << 20;        // 4 Mi fp32 or 2 Mi fp64 seeds
static __device__ __align__(256) unsigned char g_smooth_scratch[kSmoothScratchBytes];

// The array's name is a host-side stand-in in host code, not a device address: the address is asked for once per device, with that
// device current, and cached.
static lcs_status smooth_scratch_address(void **out)
{
    constexpr int kMaxDev = 64;
    static void *addr[kMaxDev] = {};
    static std::atomic<int> known[kMaxDev] = {};
    int dev = -1;
    LCS_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDev) { lcs_set_error("device ordinal %d out of range", dev); return LCS_ERR_CUDA; }
    if (!known[dev].load(std::memory_order_acquire)) {
        void *p = nullptr;
        LCS_CUDA_OK(cudaGetSymbolAddress(&p, g_smooth_scratch));
        if (!p) { lcs_set_error("cudaGetSymbolAddress returned a null address"); return LCS_ERR_CUDA; }
        addr[dev] = p;                                          // every thread that races here stores the same value
        known[dev].store(1, std::memory_order_release);
    }
    *out = addr[dev];
    return LCS_OK;
}

extern "C" lcs_status lcs_smooth_gaussian_static(int32_t dim, int32_t dtype, const int32_t ng[3], const int32_t seed_periodic[3], double sigma,
                                                 const void *field, void *out, void *cuda_stream)
{
    if ((dim != 2 && dim != 3) || !ng || !field || !out) { lcs_set_error("null argument or bad dim"); return LCS_ERR_INVALID_ARG; }
    if (dtype != LCS_F32 && dtype != LCS_F64) { lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG; }
    if (!(sigma > 0.0) || ceil(3.0 * sigma) > 64.0) { lcs_set_error("sigma must be in (0, 21.33] seed-grid cells"); return LCS_ERR_INVALID_ARG; }
    if (out == field) { lcs_set_error("field and out must be distinct buffers"); return LCS_ERR_INVALID_ARG; }
    int64_t n[3] = {1, 1, 1}, total = 1;
    for (int a = 0; a < dim; ++a) { if (ng[a] < 1) { lcs_set_error("bad seed grid"); return LCS_ERR_INVALID_ARG; } n[a] = ng[a]; total *= n[a]; }
    const size_t need = (size_t)total * lcs_esize(dtype);
    if (need > kSmoothScratchBytes) {
        lcs_set_error("lcs_smooth_gaussian_static: %lld seeds of %zu bytes exceed the static scratch of %zu bytes (max %zu seeds): use lcs_smooth_gaussian "
                      "with a work buffer", (long long)total, lcs_esize(dtype), kSmoothScratchBytes, kSmoothScratchBytes / lcs_esize(dtype));
        return LCS_ERR_INVALID_ARG;
    }
    void *work = nullptr;
    lcs_status rc = smooth_scratch_address(&work);
    if (rc != LCS_OK) return rc;
    const int64_t stride[3] = {1, n[0], n[0] * n[1]};
    const int R = (int)ceil(3.0 * sigma);
    const double inv_2s2 = 1.0 / (2.0 * sigma * sigma);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the passes of lcs_smooth_gaussian (2D: field -> work -> out; 3D: field -> out -> work -> out).  Nothing in the scratch has to
    // start at zero: every element a pass reads was written by the pass before it, whatever an earlier call left behind.
    const void *src = field;
    for (int a = 0; a < dim; ++a) {
        void *dst = ((dim - a) % 2 == 1) ? out : work;
        const int per = seed_periodic ? (seed_periodic[a] != 0) : 0;
        if (dtype == LCS_F64) LCS_LAUNCH((smooth_axis_kernel<double>), lcs_blocks(total, 256), 256, 0, st, (const double *)src, (double *)dst, total, stride[a], n[a], per, R, inv_2s2);
        else LCS_LAUNCH((smooth_axis_kernel<float>), lcs_blocks(total, 256), 256, 0, st, (const float *)src, (float *)dst, total, stride[a], n[a], per, R, inv_2s2);
        src = dst;
    }
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}

extern "C" lcs_status lcs_ridge(int32_t dim, int32_t dtype, const int32_t ng[3], const double seed_spacing[3], const int32_t seed_periodic[3],
                                double kappa_min, double s_min, const void *field, void *kappa, void *dgn, uint8_t *mask, void *cuda_stream)
{
    if ((dim != 2 && dim != 3) || !ng || !seed_spacing || !field || !kappa || !dgn || !mask) { lcs_set_error("null argument or bad dim"); return LCS_ERR_INVALID_ARG; }
    if (dtype != LCS_F32 && dtype != LCS_F64) { lcs_set_error("bad dtype"); return LCS_ERR_INVALID_ARG; }
    if (!(kappa_min >= 0.0) || !isfinite(s_min) && !(s_min < 0)) { lcs_set_error("kappa_min must be >= 0 and s_min a number"); return LCS_ERR_INVALID_ARG; }
    RidgeGrid g;
    int64_t total = 1;
    g.delta = 1e300;
    for (int a = 0; a < 3; ++a) {
        g.ng[a] = a < dim ? ng[a] : 1;
        g.per[a] = (a < dim && seed_periodic) ? (seed_periodic[a] != 0) : 0;
        g.dx[a] = a < dim ? seed_spacing[a] : 1.0;
        if (a < dim && (ng[a] < 1 || !(seed_spacing[a] > 0))) { lcs_set_error("bad seed grid on axis %d", a); return LCS_ERR_INVALID_ARG; }
        if (a < dim && g.dx[a] < g.delta) g.delta = g.dx[a];
        total *= g.ng[a];
    }
    g.kappa_min = kappa_min; g.s_min = s_min;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = lcs_blocks(total, 128);
    if (dim == 2 && dtype == LCS_F64) LCS_LAUNCH((ridge_kernel<2, double>), grid, 128, 0, st, g, (const double *)field, (double *)kappa, (double *)dgn, mask, total);
    else if (dim == 2) LCS_LAUNCH((ridge_kernel<2, float>), grid, 128, 0, st, g, (const float *)field, (float *)kappa, (float *)dgn, mask, total);
    else if (dtype == LCS_F64) LCS_LAUNCH((ridge_kernel<3, double>), grid, 128, 0, st, g, (const double *)field, (double *)kappa, (double *)dgn, mask, total);
    else LCS_LAUNCH((ridge_kernel<3, float>), grid, 128, 0, st, g, (const float *)field, (float *)kappa, (float *)dgn, mask, total);
    LCS_CUDA_OK(cudaGetLastError());
    return LCS_OK;
}
