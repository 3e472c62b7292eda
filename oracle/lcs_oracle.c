/* lcs_oracle.c -- CPU ORACLE for the LCS hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct fp64 restatement of what the hot path of arXiv 2209.13775
 * computes: point location -> space-time interpolation -> RK4 flow map -> central-
 * difference gradient -> Cauchy-Green tensor (Eq. 1.1) -> largest eigenvalue -> FTLE.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table or helper with the CUDA path
 * (paper_2209_13775_b200/csrc) and neither includes the other.
 *
 * The method is an iteration (RK4 on interpolated data) and an approximation (finite-difference
 * gradient), so the oracle follows the algorithm step by step in the paper's order; readings of
 * points where the paper is silent are the numbered "O" rules of SURVEY.md 8.2 / DESIGN.md.
 * Every function is pinned by tests/test_oracle_pins.py (pins P1-P20); nothing here is
 * "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC  (no FMA contraction: the canonical
 * face predicate must round every product and sum individually).  OpenMP over seeds only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t dim;            /* 2 | 3 */
    int32_t kind;           /* 0 Cartesian, 1 simplex */
    int32_t n[3];           /* Cartesian: nodes per axis */
    int32_t periodic[3];
    double origin[3];
    double spacing[3];
    int64_t nv, nc;         /* simplex: vertices / cells */
    const double *verts;    /* [nv][dim] */
    const int32_t *cells;   /* [nc][dim+1], any orientation */
    const int32_t *neigh;   /* [nc][dim+1], cell across the face opposite local vertex f, -1 = hull */
    int32_t ns;             /* snapshots */
    int32_t vel_f32;        /* storage type of vel: 1 = float, 0 = double (O1: widened on read) */
    const double *times;    /* [ns], uniform */
    const void *vel;        /* [ns][nv][dim]; Cartesian node = i0 + n0*(i1 + n1*i2) */
} orc_field;

/* ------------------------------------------------------------------------------------------ */
/* O1 data access: velocity stored as given, widened to fp64 on read.                          */
static inline double vel_at(const orc_field *f, int s, int64_t node, int c)
{
    int64_t nv = (f->kind == 0) ? (int64_t)f->n[0] * f->n[1] * (f->dim == 3 ? f->n[2] : 1) : f->nv;
    int64_t idx = ((int64_t)s * nv + node) * f->dim + c;
    return f->vel_f32 ? (double)((const float *)f->vel)[idx] : ((const double *)f->vel)[idx];
}

/* ------------------------------------------------------------------------------------------ */
/* O2 Cartesian location ("interpolation on Cartesian grids"; arithmetic indexing).
 * Per axis: xi = (x - origin) * inv, inv = 1/spacing computed once; i = floor(xi); w = xi - i.
 * Periodic axis: i wrapped into [0,n), upper node (i+1) mod n, stored position never wrapped.
 * Non-periodic: inside iff 0 <= xi <= n-1 (closed); i == n-1 -> i = n-2, w = 1.
 * Returns 1 if inside; lo[a]/hi[a] are the node indices of the bracketing nodes, w[a] the weight. */
static int cart_locate(const orc_field *f, const double *x, int64_t lo[3], int64_t hi[3], double w[3])
{
    for (int a = 0; a < f->dim; ++a) {
        double inv = 1.0 / f->spacing[a];
        double xi = (x[a] - f->origin[a]) * inv;
        double fl = floor(xi);
        int64_t i = (int64_t)fl;
        double wa = xi - fl;
        int64_t n = f->n[a];
        if (f->periodic[a]) {
            i = ((i % n) + n) % n;
            lo[a] = i;
            hi[a] = (i + 1) % n;
        } else {
            if (!(xi >= 0.0 && xi <= (double)(n - 1))) return 0;   /* also rejects NaN */
            if (i == n - 1) { i = n - 2; wa = 1.0; }
            lo[a] = i;
            hi[a] = i + 1;
        }
        w[a] = wa;
    }
    return 1;
}

/* cell id = i0 + nc0*(i1 + nc1*i2), nc = cells per axis (n if periodic else n-1); -1 outside. */
void orc_cart_locate(const orc_field *f, int64_t npts, const double *pos, int32_t *cell, double *wout)
{
    int d = f->dim;
    for (int64_t p = 0; p < npts; ++p) {
        int64_t lo[3] = {0, 0, 0}, hi[3]; double w[3] = {0, 0, 0};
        if (!cart_locate(f, pos + p * d, lo, hi, w)) { cell[p] = -1; continue; }
        int64_t nc0 = f->periodic[0] ? f->n[0] : f->n[0] - 1;
        int64_t nc1 = f->periodic[1] ? f->n[1] : f->n[1] - 1;
        cell[p] = (int32_t)(lo[0] + nc0 * (lo[1] + (d == 3 ? nc1 * lo[2] : 0)));
        if (wout) for (int a = 0; a < d; ++a) wout[p * d + a] = w[a];
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O2 simplex location -- the canonical face predicate (reading #8: explicit face tie-break).
 * The face's d vertices are sorted by global vertex id a<b(<c).
 *   2D: s = (bx-ax)*(py-ay) - (by-ay)*(px-ax)
 *   3D: n = (b-a) x (c-a) componentwise (uy*vz - uz*vy, ...), w = p-a, s = (nx*wx + ny*wy) + nz*wz
 * every product and sum individually rounded in fp64, left to right, no FMA.
 * side = + iff s > 0, or s == 0 and the first non-zero component of ds/dp is positive
 *   (ds/dp = (-(by-ay), bx-ax) in 2D, (nx,ny,nz) in 3D).
 * The tie rule is the symbolic perturbation p -> p + (eps, eps^2, eps^3): a point exactly on a face,
 * edge or vertex is located as that infinitesimally shifted point, which lies in general position,
 * so it has exactly one owner among the cells around it (the rule "tie -> + side of the id-sorted
 * face" proposed in SURVEY.md 8.2 is consistent across a face but not around an edge: pin P9 found
 * points with 0 and 2 owners).  Both cells sharing a face evaluate the identical expression, so
 * exactly one of them accepts p with respect to that face: no gaps and no overlaps.               */
static inline int face_side(const orc_field *f, const int32_t *fv /* d sorted vertex ids */, const double *p)
{
    if (f->dim == 2) {
        const double *a = f->verts + 2 * (int64_t)fv[0], *b = f->verts + 2 * (int64_t)fv[1];
        double ex = b[0] - a[0], ey = b[1] - a[1];
        double s = ex * (p[1] - a[1]) - ey * (p[0] - a[0]);
        if (s != 0.0) return s > 0.0;
        if (ey != 0.0) return -ey > 0.0;
        return ex > 0.0;
    } else {
        const double *a = f->verts + 3 * (int64_t)fv[0], *b = f->verts + 3 * (int64_t)fv[1],
                     *c = f->verts + 3 * (int64_t)fv[2];
        double ux = b[0] - a[0], uy = b[1] - a[1], uz = b[2] - a[2];
        double vx = c[0] - a[0], vy = c[1] - a[1], vz = c[2] - a[2];
        double nx = uy * vz - uz * vy;
        double ny = uz * vx - ux * vz;
        double nz = ux * vy - uy * vx;
        double wx = p[0] - a[0], wy = p[1] - a[1], wz = p[2] - a[2];
        double s = (nx * wx + ny * wy) + nz * wz;
        if (s != 0.0) return s > 0.0;
        if (nx != 0.0) return nx > 0.0;
        if (ny != 0.0) return ny > 0.0;
        return nz > 0.0;
    }
}

/* sorted vertex ids of the face of cell c opposite its local vertex fidx */
static inline void face_verts(const orc_field *f, int64_t c, int fidx, int32_t *fv)
{
    int d = f->dim, k = 0;
    const int32_t *cv = f->cells + c * (d + 1);
    for (int j = 0; j <= d; ++j) if (j != fidx) fv[k++] = cv[j];
    /* insertion sort of 2 or 3 ids */
    for (int i = 1; i < d; ++i) {
        int32_t key = fv[i]; int j = i - 1;
        while (j >= 0 && fv[j] > key) { fv[j + 1] = fv[j]; --j; }
        fv[j + 1] = key;
    }
}

/* index of the first face (local order 0..d) whose side test fails for p, or -1 if c accepts p:
 * c contains p iff for each face, side(face,p) == side(face, opposite vertex of c).            */
static inline int first_failing_face(const orc_field *f, int64_t c, const double *p)
{
    int d = f->dim;
    const int32_t *cv = f->cells + c * (d + 1);
    for (int j = 0; j <= d; ++j) {
        int32_t fv[3];
        face_verts(f, c, j, fv);
        int sp = face_side(f, fv, p);
        int so = face_side(f, fv, f->verts + (int64_t)d * cv[j]);
        if (sp != so) return j;
    }
    return -1;
}

/* Brute force = the definition: lowest-index accepting cell or -1; count = number of accepting cells. */
static int64_t simplex_locate_brute1(const orc_field *f, const double *p, int32_t *count)
{
    int64_t found = -1; int32_t cnt = 0;
    for (int64_t c = 0; c < f->nc; ++c)
        if (first_failing_face(f, c, p) < 0) { if (found < 0) found = c; ++cnt; }
    if (count) *count = cnt;
    return found;
}

void orc_simplex_locate_brute(const orc_field *f, int64_t npts, const double *pos, int32_t *cell, int32_t *count)
{
    int d = f->dim;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t p = 0; p < npts; ++p) {
        int32_t cnt;
        cell[p] = (int32_t)simplex_locate_brute1(f, pos + p * d, &cnt);
        if (count) count[p] = cnt;
    }
}

/* validity check used where several answers are acceptable (points within rounding of an edge or a
 * vertex, where the signs of mathematically-zero s values are rounding noise): does `cell` accept p? */
void orc_simplex_accepts(const orc_field *f, int64_t npts, const double *pos, const int32_t *cell, int32_t *ok)
{
    for (int64_t p = 0; p < npts; ++p)
        ok[p] = (cell[p] >= 0 && cell[p] < f->nc) ? (first_failing_face(f, cell[p], pos + p * f->dim) < 0) : 0;
}

/* Fast mode ("efficient local cell search", reading #6): walk from a start cell across
 * the first failing face in local-face order; a hull face (-1 neighbour) => outside (reading #11);
 * hop cap 4*nc^(1/d)+64, then fall back to brute force.  Same canonical predicate as the definition. */
static int64_t simplex_walk(const orc_field *f, int64_t start, const double *p)
{
    int d = f->dim;
    int64_t cap = (int64_t)(4.0 * pow((double)f->nc, 1.0 / d)) + 64;
    int64_t c = start;
    if (c < 0 || c >= f->nc) return simplex_locate_brute1(f, p, NULL);
    for (int64_t hop = 0; hop < cap; ++hop) {
        int j = first_failing_face(f, c, p);
        if (j < 0) return c;
        int64_t nb = f->neigh[c * (d + 1) + j];
        if (nb < 0) return -1;
        c = nb;
    }
    return simplex_locate_brute1(f, p, NULL);
}

void orc_simplex_locate_walk(const orc_field *f, int64_t npts, const double *pos, const int32_t *start, int32_t *cell)
{
    int d = f->dim;
    #pragma omp parallel for schedule(dynamic, 256)
    for (int64_t p = 0; p < npts; ++p)
        cell[p] = (int32_t)simplex_walk(f, start ? start[p] : 0, pos + p * d);
}

/* Face-neighbour table: two cells are neighbours across a face iff the face's sorted vertex ids
 * coincide.  Sort all (face key, cell, local face) records; equal adjacent keys pair up.
 * Returns 0, or 3 (mesh error) if some face is shared by more than two cells.                   */
typedef struct { int32_t k[3]; int32_t cell; int32_t face; } face_rec;
static int face_cmp(const void *x, const void *y)
{
    const face_rec *a = (const face_rec *)x, *b = (const face_rec *)y;
    for (int i = 0; i < 3; ++i) if (a->k[i] != b->k[i]) return a->k[i] < b->k[i] ? -1 : 1;
    return 0;
}
int orc_simplex_build_neighbours(int32_t dim, int64_t nc, const int32_t *cells, int32_t *neigh)
{
    orc_field tmp; memset(&tmp, 0, sizeof tmp); tmp.dim = dim; tmp.cells = cells;
    int64_t nf = nc * (dim + 1);
    face_rec *r = (face_rec *)malloc(sizeof(face_rec) * (size_t)nf);
    if (!r) return 4;
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j <= dim; ++j) {
            face_rec *q = r + c * (dim + 1) + j;
            q->k[2] = -1;
            face_verts(&tmp, c, j, q->k);
            q->cell = (int32_t)c; q->face = j;
        }
    qsort(r, (size_t)nf, sizeof(face_rec), face_cmp);
    for (int64_t i = 0; i < nf; ++i) neigh[i] = -1;
    int rc = 0;
    for (int64_t i = 0; i < nf;) {
        int64_t j = i + 1;
        while (j < nf && face_cmp(r + i, r + j) == 0) ++j;
        if (j - i == 2) {
            neigh[(int64_t)r[i].cell * (dim + 1) + r[i].face] = r[i + 1].cell;
            neigh[(int64_t)r[i + 1].cell * (dim + 1) + r[i + 1].face] = r[i].cell;
        } else if (j - i > 2) rc = 3;
        i = j;
    }
    free(r);
    return rc;
}

/* ------------------------------------------------------------------------------------------ */
/* O3 interpolation (space and time interpolation, nominally two frames, linear
 * in time; per-grid-type spatial interpolation).
 * Time: s = clamp(floor((t - times[0]) / dt), 0, ns-2); tau = (t - times[s]) / (times[s+1] - times[s]),
 * tau NOT clamped.  u(x,t) = u_s + tau*(u_{s+1} - u_s) after the spatial step on each snapshot.   */
static inline double lerp(double a, double b, double w) { return a + w * (b - a); }

static void time_bracket(const orc_field *f, double t, int *s, double *tau)
{
    double dt = f->times[1] - f->times[0];
    double q = floor((t - f->times[0]) / dt);
    int si = (q < 0.0) ? 0 : (q > (double)(f->ns - 2) ? f->ns - 2 : (int)q);
    *s = si;
    *tau = (t - f->times[si]) / (f->times[si + 1] - f->times[si]);
}

/* bi/trilinear, nested-lerp order x, then y, then z (reading #4) */
static void cart_space_interp(const orc_field *f, int s, const int64_t lo[3], const int64_t hi[3],
                              const double w[3], double *u)
{
    int d = f->dim;
    int64_t n0 = f->n[0], n1 = f->n[1];
    for (int c = 0; c < d; ++c) {
        if (d == 2) {
            double a0 = lerp(vel_at(f, s, lo[0] + n0 * lo[1], c), vel_at(f, s, hi[0] + n0 * lo[1], c), w[0]);
            double a1 = lerp(vel_at(f, s, lo[0] + n0 * hi[1], c), vel_at(f, s, hi[0] + n0 * hi[1], c), w[0]);
            u[c] = lerp(a0, a1, w[1]);
        } else {
            double b[2];
            for (int kz = 0; kz < 2; ++kz) {
                int64_t k = kz ? hi[2] : lo[2];
                double a0 = lerp(vel_at(f, s, lo[0] + n0 * (lo[1] + n1 * k), c),
                                 vel_at(f, s, hi[0] + n0 * (lo[1] + n1 * k), c), w[0]);
                double a1 = lerp(vel_at(f, s, lo[0] + n0 * (hi[1] + n1 * k), c),
                                 vel_at(f, s, hi[0] + n0 * (hi[1] + n1 * k), c), w[0]);
                b[kz] = lerp(a0, a1, w[1]);
            }
            u[c] = lerp(b[0], b[1], w[2]);
        }
    }
}

/* barycentric (P1) weights of p in cell c, relative to vertex 0 (reading #5): lambda_i = s_i / s_total,
 * s_i = signed volume with vertex i replaced by p.  Not the canonical predicate: values only.       */
static void bary_weights(const orc_field *f, int64_t c, const double *p, double *lam)
{
    int d = f->dim;
    const int32_t *cv = f->cells + c * (d + 1);
    const double *v0 = f->verts + (int64_t)d * cv[0];
    if (d == 2) {
        const double *v1 = f->verts + 2 * (int64_t)cv[1], *v2 = f->verts + 2 * (int64_t)cv[2];
        double e1x = v1[0] - v0[0], e1y = v1[1] - v0[1];
        double e2x = v2[0] - v0[0], e2y = v2[1] - v0[1];
        double px = p[0] - v0[0], py = p[1] - v0[1];
        double tot = e1x * e2y - e1y * e2x;
        lam[1] = (px * e2y - py * e2x) / tot;      /* vertex 1 replaced by p */
        lam[2] = (e1x * py - e1y * px) / tot;      /* vertex 2 replaced by p */
        lam[0] = 1.0 - lam[1] - lam[2];
    } else {
        const double *v1 = f->verts + 3 * (int64_t)cv[1], *v2 = f->verts + 3 * (int64_t)cv[2],
                     *v3 = f->verts + 3 * (int64_t)cv[3];
        double e1[3], e2[3], e3[3], q[3];
        for (int i = 0; i < 3; ++i) { e1[i] = v1[i] - v0[i]; e2[i] = v2[i] - v0[i]; e3[i] = v3[i] - v0[i]; q[i] = p[i] - v0[i]; }
        #define DET3(a, b, c) ((a)[0] * ((b)[1] * (c)[2] - (b)[2] * (c)[1]) - (a)[1] * ((b)[0] * (c)[2] - (b)[2] * (c)[0]) + (a)[2] * ((b)[0] * (c)[1] - (b)[1] * (c)[0]))
        double tot = DET3(e1, e2, e3);
        lam[1] = DET3(q, e2, e3) / tot;
        lam[2] = DET3(e1, q, e3) / tot;
        lam[3] = DET3(e1, e2, q) / tot;
        lam[0] = 1.0 - lam[1] - lam[2] - lam[3];
        #undef DET3
    }
}

/* u(x,t); *cell is the tracer's current cell (simplex: in/out, walk start; Cartesian: unused).
 * Returns 1 and fills u if x is inside the mesh, else 0 ("no value": triggers exit).               */
static int velocity(const orc_field *f, const double *x, double t, int64_t *cell, double *u)
{
    int s; double tau;
    int d = f->dim;
    time_bracket(f, t, &s, &tau);
    double ua[3], ub[3];
    if (f->kind == 0) {
        int64_t lo[3], hi[3]; double w[3];
        if (!cart_locate(f, x, lo, hi, w)) return 0;
        cart_space_interp(f, s, lo, hi, w, ua);
        cart_space_interp(f, s + 1, lo, hi, w, ub);
    } else {
        int64_t c = simplex_walk(f, *cell, x);
        if (c < 0) return 0;
        *cell = c;
        double lam[4];
        bary_weights(f, c, x, lam);
        const int32_t *cv = f->cells + c * (d + 1);
        for (int k = 0; k < d; ++k) {
            double sa = 0.0, sb = 0.0;
            for (int i = 0; i <= d; ++i) {
                sa = sa + lam[i] * vel_at(f, s, cv[i], k);
                sb = sb + lam[i] * vel_at(f, s + 1, cv[i], k);
            }
            ua[k] = sa; ub[k] = sb;
        }
    }
    for (int k = 0; k < d; ++k) u[k] = ua[k] + tau * (ub[k] - ua[k]);
    return 1;
}

/* test hook: velocity at arbitrary points and one time */
void orc_velocity(const orc_field *f, int64_t npts, const double *pos, double t, const int32_t *start,
                  double *u, int32_t *inside)
{
    int d = f->dim;
    #pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < npts; ++p) {
        int64_t c = start ? start[p] : 0;
        double uu[3] = {0, 0, 0};
        int ok = velocity(f, pos + p * d, t, &c, uu);
        inside[p] = ok;
        for (int k = 0; k < d; ++k) u[p * d + k] = ok ? uu[k] : NAN;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O4 RK4 flow map (Eq. 1.2; classical 4th-order Runge-Kutta with four space-time
 * evaluations per step; exit handling PAPER.md:65, reading #9/#10).
 * N = llround((tf-t0)/h).  Step n: ta = t0 + n*h, tb = t0 + (n+0.5)*h, tc = t0 + (n+1)*h (products).
 * k1=u(x,ta); k2=u(x+(h/2)k1,tb); k3=u(x+(h/2)k2,tb); k4=u(x+h*k3,tc); x += (h/6)(k1+2k2+2k3+k4).
 * Any of the four evaluation points outside: x keeps its start-of-step value, flag 1, exit_step n.
 * Seed outside at t0: flag 2, flow map = seed, exit_step 0.  h<0 = backward time.
 * cell0: simplex only, the seed's cell from orc_simplex_locate_* (-1 = outside).
 * traj (optional): [n_rec][npts][dim] positions after every rec_every steps (for e_D(t)). */
void orc_advect(const orc_field *f, int64_t npts, const double *seeds, double t0, double tf, double h,
                const int32_t *cell0, double *flowmap, uint8_t *flag, int32_t *exit_step,
                int32_t rec_every, double *traj)
{
    int d = f->dim;
    int64_t N = llround((tf - t0) / h);
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t p = 0; p < npts; ++p) {
        double x[3] = {0, 0, 0};
        for (int k = 0; k < d; ++k) x[k] = seeds[p * d + k];
        int64_t cell = 0;
        uint8_t fl = 0; int32_t es = (int32_t)N;
        if (f->kind == 1) {
            cell = cell0 ? cell0[p] : simplex_locate_brute1(f, x, NULL);
            if (cell < 0) { fl = 2; es = 0; }
        } else {
            int64_t lo[3], hi[3]; double w[3];
            if (!cart_locate(f, x, lo, hi, w)) { fl = 2; es = 0; }
        }
        for (int64_t n = 0; n < N && fl == 0; ++n) {
            double ta = t0 + (double)n * h, tb = t0 + ((double)n + 0.5) * h, tc = t0 + ((double)n + 1.0) * h;
            double k1[3], k2[3], k3[3], k4[3], y[3];
            int64_t c = cell;
            int ok = velocity(f, x, ta, &c, k1);
            if (ok) { for (int k = 0; k < d; ++k) y[k] = x[k] + (h / 2) * k1[k]; ok = velocity(f, y, tb, &c, k2); }
            if (ok) { for (int k = 0; k < d; ++k) y[k] = x[k] + (h / 2) * k2[k]; ok = velocity(f, y, tb, &c, k3); }
            if (ok) { for (int k = 0; k < d; ++k) y[k] = x[k] + h * k3[k];       ok = velocity(f, y, tc, &c, k4); }
            if (!ok) { fl = 1; es = (int32_t)n; break; }
            for (int k = 0; k < d; ++k) x[k] = x[k] + (h / 6) * (k1[k] + 2 * k2[k] + 2 * k3[k] + k4[k]);
            cell = c;
            if (traj && rec_every > 0 && (n + 1) % rec_every == 0)
                for (int k = 0; k < d; ++k) traj[(((n + 1) / rec_every - 1) * npts + p) * d + k] = x[k];
        }
        if (traj && rec_every > 0 && fl != 0)      /* frozen tracers keep their last position */
            for (int64_t r = (fl == 2 ? 0 : es / rec_every); r < N / rec_every; ++r)
                for (int k = 0; k < d; ++k) traj[(r * npts + p) * d + k] = x[k];
        for (int k = 0; k < d; ++k) flowmap[p * d + k] = x[k];
        if (flag) flag[p] = fl;
        if (exit_step) exit_step[p] = es;
    }
}

/* ---- O12 (row f4, second part): multi-step integrator ------------------------------------------------------
 * The Flow Map filter can use "Runge-Kutta (single-step)" or "Adams-Bashforth (multi-step)" integrators;
 * no order or start-up is given.  Reading (#31): 4-step Adams-Bashforth, started with three classical RK4
 * steps (rule O4).  f_n = u(x_n, t_n), t_n = t0 + n h (by multiplication);
 *   n >= 3:  x_{n+1} = x_n + (h / 24) (55 f_n - 59 f_{n-1} + 37 f_{n-2} - 9 f_{n-3}).
 * One velocity evaluation per step after the start-up.  Exit: an evaluation point outside the domain => x keeps its
 * start-of-step value, flag 1, exit_step n (as O4; an AB step can carry x_{n+1} itself outside, which the next step's
 * evaluation then reports).  Same argument conventions as orc_advect.                                              */
void orc_advect_ab4(const orc_field *f, int64_t npts, const double *seeds, double t0, double tf, double h,
                    const int32_t *cell0, double *flowmap, uint8_t *flag, int32_t *exit_step)
{
    int d = f->dim;
    int64_t N = llround((tf - t0) / h);
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t p = 0; p < npts; ++p) {
        double x[3] = {0, 0, 0}, hist[3][3];             /* hist[0] = f_{n-1}, hist[1] = f_{n-2}, hist[2] = f_{n-3} */
        for (int k = 0; k < d; ++k) x[k] = seeds[p * d + k];
        int64_t cell = 0;
        uint8_t fl = 0; int32_t es = (int32_t)N;
        if (f->kind == 1) {
            cell = cell0 ? cell0[p] : simplex_locate_brute1(f, x, NULL);
            if (cell < 0) { fl = 2; es = 0; }
        } else {
            int64_t lo[3], hi[3]; double w[3];
            if (!cart_locate(f, x, lo, hi, w)) { fl = 2; es = 0; }
        }
        for (int64_t n = 0; n < N && fl == 0; ++n) {
            double ta = t0 + (double)n * h, tb = t0 + ((double)n + 0.5) * h, tc = t0 + ((double)n + 1.0) * h;
            double k1[3], k2[3], k3[3], k4[3], y[3];
            int64_t c = cell;
            int ok = velocity(f, x, ta, &c, k1);            /* f_n */
            if (ok && n < 3) {
                for (int k = 0; k < d; ++k) y[k] = x[k] + (h / 2) * k1[k];
                ok = velocity(f, y, tb, &c, k2);
                if (ok) { for (int k = 0; k < d; ++k) y[k] = x[k] + (h / 2) * k2[k]; ok = velocity(f, y, tb, &c, k3); }
                if (ok) { for (int k = 0; k < d; ++k) y[k] = x[k] + h * k3[k];       ok = velocity(f, y, tc, &c, k4); }
            }
            if (!ok) { fl = 1; es = (int32_t)n; break; }
            if (n < 3) {
                for (int k = 0; k < d; ++k) x[k] = x[k] + (h / 6) * (k1[k] + 2 * k2[k] + 2 * k3[k] + k4[k]);
            } else {
                for (int k = 0; k < d; ++k)
                    x[k] = x[k] + (h / 24) * (55 * k1[k] - 59 * hist[0][k] + 37 * hist[1][k] - 9 * hist[2][k]);
            }
            for (int k = 0; k < d; ++k) { hist[2][k] = hist[1][k]; hist[1][k] = hist[0][k]; hist[0][k] = k1[k]; }
            cell = c;
        }
        for (int k = 0; k < d; ++k) flowmap[p * d + k] = x[k];
        if (flag) flag[p] = fl;
        if (exit_step) exit_step[p] = es;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* O7 largest eigenvalue of a symmetric matrix, closed form.
 * 2x2: lambda = (C11+C22)/2 + sqrt(((C11-C22)/2)^2 + C12^2).
 * 3x3: trigonometric form: q = tr/3; p1 = C12^2+C13^2+C23^2; p2 = sum (Cii-q)^2 + 2 p1; p2 == 0 -> q;
 *      p = sqrt(p2/6); B = (C - qI)/p; r = clamp(det B / 2, -1, 1); lambda = q + 2 p cos(acos(r)/3). */
double orc_eigmax_sym2(double c11, double c12, double c22)
{
    double hd = 0.5 * (c11 - c22);
    return 0.5 * (c11 + c22) + sqrt(hd * hd + c12 * c12);
}
double orc_eigmax_sym3(double c11, double c12, double c13, double c22, double c23, double c33)
{
    double q = (c11 + c22 + c33) / 3.0;
    double p1 = c12 * c12 + c13 * c13 + c23 * c23;
    double p2 = (c11 - q) * (c11 - q) + (c22 - q) * (c22 - q) + (c33 - q) * (c33 - q) + 2.0 * p1;
    if (p2 == 0.0) return q;
    double p = sqrt(p2 / 6.0);
    double b11 = (c11 - q) / p, b22 = (c22 - q) / p, b33 = (c33 - q) / p;
    double b12 = c12 / p, b13 = c13 / p, b23 = c23 / p;
    double det = b11 * (b22 * b33 - b23 * b23) - b12 * (b12 * b33 - b23 * b13) + b13 * (b12 * b23 - b22 * b13);
    double r = det / 2.0;
    if (r < -1.0) r = -1.0;
    if (r > 1.0) r = 1.0;
    return q + 2.0 * p * cos(acos(r) / 3.0);
}

/* O5 + O6 + O7: central-difference flow-map gradient on the structured seed grid,
 * Cauchy-Green tensor C = G^T G with G_ab = dF_a/dx_b (Eq. 1.1; reading #14), largest
 * eigenvalue, FTLE = ln(lambda_max) / (2|T|) (reading #1).
 * Seed index (i,j,k), axis 0 fastest.  A neighbour is valid if inside the grid (or reached by periodic
 * wrap: +-period[b] added to its F_b only) and its exit_flag == 0.  Both valid: central; one valid and
 * the seed itself valid: first-order one-sided (status bit 1); seed invalid or neither neighbour valid
 * on some axis: C, FTLE = NaN, status bit 0 (reading #12).
 * cg: [n][3] (C11,C12,C22) or [n][6] (C11,C12,C13,C22,C23,C33); may be NULL.                        */
void orc_cg_ftle(int32_t dim, const int32_t *ng, const double *dx, const int32_t *sper, const double *period,
                 const double *F, const uint8_t *flag, double T, double *cg, double *ftle, uint8_t *status)
{
    int64_t n0 = ng[0], n1 = ng[1], n2 = (dim == 3) ? ng[2] : 1;
    int ncg = (dim == 2) ? 3 : 6;
    int64_t stride[3] = {1, n0, n0 * n1};
    #pragma omp parallel for schedule(static)
    for (int64_t idx = 0; idx < n0 * n1 * n2; ++idx) {
        int64_t ijk[3] = {idx % n0, (idx / n0) % n1, idx / (n0 * n1)};
        double G[3][3];
        uint8_t st = 0;
        int self_ok = flag ? (flag[idx] == 0) : 1;
        if (!self_ok) st |= 1;
        for (int b = 0; b < dim && !(st & 1); ++b) {
            int64_t nb = ng[b];
            int64_t ip = ijk[b] + 1, im = ijk[b] - 1;
            double shp = 0.0, shm = 0.0;
            int okp = 1, okm = 1;
            if (ip >= nb) { if (sper[b]) { ip -= nb; shp = period[b]; } else okp = 0; }
            if (im < 0)   { if (sper[b]) { im += nb; shm = -period[b]; } else okm = 0; }
            int64_t jp = idx + (ip - ijk[b]) * stride[b], jm = idx + (im - ijk[b]) * stride[b];
            if (okp && flag && flag[jp] != 0) okp = 0;
            if (okm && flag && flag[jm] != 0) okm = 0;
            for (int a = 0; a < dim; ++a) {
                double Fp = okp ? F[jp * dim + a] + (a == b ? shp : 0.0) : 0.0;
                double Fm = okm ? F[jm * dim + a] + (a == b ? shm : 0.0) : 0.0;
                double F0 = F[idx * dim + a];
                if (okp && okm)      G[a][b] = (Fp - Fm) / (2.0 * dx[b]);
                else if (okp)        G[a][b] = (Fp - F0) / dx[b];
                else if (okm)        G[a][b] = (F0 - Fm) / dx[b];
            }
            if (!okp && !okm) st |= 1;
            else if (!(okp && okm)) st |= 2;
        }
        double C[6];
        double lam;
        if (st & 1) {
            for (int i = 0; i < ncg; ++i) C[i] = NAN;
            lam = NAN;
        } else if (dim == 2) {
            C[0] = G[0][0] * G[0][0] + G[1][0] * G[1][0];
            C[1] = G[0][0] * G[0][1] + G[1][0] * G[1][1];
            C[2] = G[0][1] * G[0][1] + G[1][1] * G[1][1];
            lam = orc_eigmax_sym2(C[0], C[1], C[2]);
        } else {
            int m = 0;
            for (int b = 0; b < 3; ++b)
                for (int c = b; c < 3; ++c) {
                    double s = 0.0;
                    for (int a = 0; a < 3; ++a) s = s + G[a][b] * G[a][c];
                    C[m++] = s;
                }
            lam = orc_eigmax_sym3(C[0], C[1], C[2], C[3], C[4], C[5]);
        }
        if (cg) for (int i = 0; i < ncg; ++i) cg[idx * ncg + i] = C[i];
        ftle[idx] = (st & 1) ? NAN : log(lam) / (2.0 * fabs(T));
        if (status) status[idx] = st;
    }
}

/* ---- O8 (row f2): full eigen-decomposition of the Cauchy-Green tensor ---------------------------------------
 * The Cauchy-Green filter attaches "eigenvalues and eigenvectors" of C to the seed points; the
 * eigenvectors are what hyperbolic-LCS criteria (strainlines) need.  The paper gives no algorithm.
 * Reading (#27): classical cyclic Jacobi on the symmetric d x d matrix in fp64 (the closed forms are
 * ill-conditioned for the small eigenvalues): sweep the pairs (0,1), (0,2), (1,2), rotate away each off-diagonal
 * entry with the stable tangent formula t = sgn(theta) / (|theta| + sqrt(theta^2 + 1)), theta = (a_qq - a_pp) / (2 a_pq);
 * stop when every off-diagonal entry is exactly zero or after 50 sweeps.  Eigenvalues ascending; row i of evec is
 * the unit eigenvector of eval[i], sign fixed so that its component of largest magnitude (first on ties) is positive.
 * Any non-finite input gives NaN everywhere.  cg: [n][3] (C11,C12,C22) or [n][6] (C11,C12,C13,C22,C23,C33).           */
static void jacobi_sym(int d, double a[3][3], double v[3][3])
{
    for (int i = 0; i < d; ++i)
        for (int j = 0; j < d; ++j) v[i][j] = (i == j) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 50; ++sweep) {
        double off = 0.0;
        for (int p = 0; p < d; ++p)
            for (int q = p + 1; q < d; ++q) off += fabs(a[p][q]);
        if (off == 0.0) break;
        for (int p = 0; p < d; ++p)
            for (int q = p + 1; q < d; ++q) {
                double apq = a[p][q];
                if (apq == 0.0) continue;
                double theta = (a[q][q] - a[p][p]) / (2.0 * apq);
                double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                if (!isfinite(theta)) t = 0.0;          /* a_pq negligible against the diagonal gap */
                double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                a[p][p] -= t * apq;
                a[q][q] += t * apq;
                a[p][q] = a[q][p] = 0.0;
                for (int r = 0; r < d; ++r) {
                    if (r != p && r != q) {
                        double arp = a[r][p], arq = a[r][q];
                        a[r][p] = a[p][r] = c * arp - s * arq;
                        a[r][q] = a[q][r] = s * arp + c * arq;
                    }
                    double vrp = v[r][p], vrq = v[r][q];   /* columns of v are the eigenvectors */
                    v[r][p] = c * vrp - s * vrq;
                    v[r][q] = s * vrp + c * vrq;
                }
            }
    }
}

void orc_cg_eigen(int32_t dim, int64_t n, const double *cg, double *evals, double *evecs)
{
    const int d = dim, ncg = dim == 2 ? 3 : 6;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double *c = cg + i * ncg;
        double *ev = evals + i * d, *vv = evecs + i * d * d;
        int finite = 1;
        for (int k = 0; k < ncg; ++k) finite = finite && isfinite(c[k]);
        if (!finite) {
            for (int k = 0; k < d; ++k) ev[k] = NAN;
            for (int k = 0; k < d * d; ++k) vv[k] = NAN;
            continue;
        }
        double a[3][3], v[3][3];
        if (d == 2) { a[0][0] = c[0]; a[0][1] = a[1][0] = c[1]; a[1][1] = c[2]; }
        else { a[0][0] = c[0]; a[0][1] = a[1][0] = c[1]; a[0][2] = a[2][0] = c[2]; a[1][1] = c[3]; a[1][2] = a[2][1] = c[4]; a[2][2] = c[5]; }
        jacobi_sym(d, a, v);
        int order[3] = {0, 1, 2};
        for (int x = 0; x < d; ++x)                      /* ascending, stable */
            for (int y = x + 1; y < d; ++y)
                if (a[order[y]][order[y]] < a[order[x]][order[x]]) { int t = order[x]; order[x] = order[y]; order[y] = t; }
        for (int k = 0; k < d; ++k) {
            int col = order[k], big = 0;
            ev[k] = a[col][col];
            for (int r = 1; r < d; ++r)
                if (fabs(v[r][col]) > fabs(v[big][col])) big = r;
            double sg = v[big][col] < 0.0 ? -1.0 : 1.0;
            for (int r = 0; r < d; ++r) vv[k * d + r] = sg * v[r][col];
        }
    }
}

/* ---- O9 (row f3): Cauchy-Green tensor from auxiliary points -------------------------------------------------
 * "a structured grid of auxiliary points can be placed around each seed point" and the Cauchy-Green
 * filter can use them "for the computation of the flow map gradient" instead of the neighbouring seeds.
 * Reading (#28): 2 d auxiliary tracers per seed, released at x0 + delta_b e_b and x0 - delta_b e_b;
 * Faux[i][2 b][.] / Faux[i][2 b + 1][.] are their final positions; G_ab = (F_a(+b) - F_a(-b)) / (2 delta_b), always
 * central; if any of the 2 d auxiliary tracers of a seed has a non-zero exit flag: C, FTLE = NaN, status bit 0.
 * C, lambda_max and FTLE then follow O6-O7.                                                                    */
void orc_cg_ftle_aux(int32_t dim, int64_t n, const double *delta, const double *Faux, const uint8_t *flag_aux, double T,
                     double *cg, double *ftle, uint8_t *status)
{
    const int d = dim, ncg = dim == 2 ? 3 : 6;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double G[3][3], C[6], lam;
        uint8_t st = 0;
        for (int k = 0; k < 2 * d; ++k)
            if (flag_aux && flag_aux[i * 2 * d + k] != 0) st = 1;
        for (int b = 0; b < d; ++b)
            for (int a = 0; a < d; ++a) {
                double Fp = Faux[(i * 2 * d + 2 * b) * d + a], Fm = Faux[(i * 2 * d + 2 * b + 1) * d + a];
                G[a][b] = (Fp - Fm) / (2.0 * delta[b]);
            }
        if (st) {
            for (int k = 0; k < ncg; ++k) C[k] = NAN;
            lam = NAN;
        } else if (d == 2) {
            C[0] = G[0][0] * G[0][0] + G[1][0] * G[1][0];
            C[1] = G[0][0] * G[0][1] + G[1][0] * G[1][1];
            C[2] = G[0][1] * G[0][1] + G[1][1] * G[1][1];
            lam = orc_eigmax_sym2(C[0], C[1], C[2]);
        } else {
            int m = 0;
            for (int b = 0; b < 3; ++b)
                for (int c = b; c < 3; ++c) {
                    double s = 0.0;
                    for (int a = 0; a < 3; ++a) s = s + G[a][b] * G[a][c];
                    C[m++] = s;
                }
            lam = orc_eigmax_sym3(C[0], C[1], C[2], C[3], C[4], C[5]);
        }
        if (cg) for (int k = 0; k < ncg; ++k) cg[i * ncg + k] = C[k];
        ftle[i] = st ? NAN : log(lam) / (2.0 * fabs(T));
        if (status) status[i] = st;
    }
}

/* ---- O11 (row f4, first part): Gaussian smoothing of the FTLE field ------------------------------------------
 * The LCS filter smooths the FTLE field with a Gaussian before extracting ridges; no parameters given.
 * Reading (#30): one normalised 1D convolution per axis, axis 0 first, on the structured seed grid:
 *   out(i) = sum_k w_k f(i+k) / sum_k w_k over |k| <= R = ceil(3 sigma) with f(i+k) finite and inside the grid
 *   (index wrapped on a periodic axis), w_k = exp(-k^2 / (2 sigma^2)), sigma in seed-grid cells;
 * a NaN centre stays NaN (undefined seeds are not filled in), NaN neighbours are skipped.  fp64 throughout.       */
void orc_smooth_gaussian(int32_t dim, const int32_t *ng, const int32_t *sper, double sigma, const double *in, double *out)
{
    int64_t n[3] = {ng[0], ng[1], dim == 3 ? ng[2] : 1};
    int64_t total = n[0] * n[1] * n[2], stride[3] = {1, n[0], n[0] * n[1]};
    int R = (int)ceil(3.0 * sigma);
    double *a = (double *)malloc(sizeof(double) * (size_t)total), *b = (double *)malloc(sizeof(double) * (size_t)total);
    memcpy(a, in, sizeof(double) * (size_t)total);
    for (int ax = 0; ax < dim; ++ax) {
#pragma omp parallel for schedule(static)
        for (int64_t idx = 0; idx < total; ++idx) {
            int64_t i = (idx / stride[ax]) % n[ax];
            if (!isfinite(a[idx])) { b[idx] = a[idx]; continue; }
            double num = 0.0, den = 0.0;
            for (int k = -R; k <= R; ++k) {
                int64_t j = i + k;
                if (sper[ax]) j = ((j % n[ax]) + n[ax]) % n[ax];
                else if (j < 0 || j >= n[ax]) continue;
                double v = a[idx + (j - i) * stride[ax]];
                if (!isfinite(v)) continue;
                double w = exp(-(double)(k * k) / (2.0 * sigma * sigma));
                num += w * v;
                den += w;
            }
            b[idx] = num / den;
        }
        double *t = a; a = b; b = t;
    }
    memcpy(out, a, sizeof(double) * (size_t)total);
    free(a); free(b);
}

/* ---- O13 (row f4, third part): ridges of the (smoothed) FTLE field ---------------------------------------------
 * The LCS filter extracts "C-ridges" of the smoothed FTLE field; the paper gives no definition.
 * Reading (#32): the second-derivative ridge of the FTLE literature (the paper's ref [29]): with g the gradient
 * and H the Hessian of the field s, n the unit eigenvector of the SMALLEST eigenvalue kappa of H, a ridge point has
 * kappa < 0 and g . n = 0.  On the seed grid, per seed:
 *   g_a  = (s(+a) - s(-a)) / (2 dx_a);  H_aa = (s(+a) - 2 s + s(-a)) / dx_a^2;
 *   H_ab = (s(+a+b) - s(+a-b) - s(-a+b) + s(-a-b)) / (4 dx_a dx_b);   neighbours wrapped on periodic axes;
 *   (kappa, n) by the Jacobi iteration of O8 (sign of n: component of largest magnitude positive);  d = g . n;
 *   mask = 1 iff kappa < -kappa_min and s >= s_min and |d| <= |kappa| * delta / 2,  delta = min_a dx_a
 *   (to first order |d| / |kappa| is the distance to the ridge along n: the ridge passes within half a cell).
 * A seed whose stencil (the 3^d block) leaves the grid on a non-periodic axis or contains a non-finite value gets
 * kappa = d = NaN, mask = 0.                                                                                       */
void orc_ridge(int32_t dim, const int32_t *ng, const double *dx, const int32_t *sper, double kappa_min, double s_min,
               const double *field, double *kappa, double *dgn, uint8_t *mask)
{
    int64_t n[3] = {ng[0], ng[1], dim == 3 ? ng[2] : 1};
    int64_t total = n[0] * n[1] * n[2], stride[3] = {1, n[0], n[0] * n[1]};
    double delta = dx[0];
    for (int a = 1; a < dim; ++a) if (dx[a] < delta) delta = dx[a];
#pragma omp parallel for schedule(static)
    for (int64_t idx = 0; idx < total; ++idx) {
        int64_t ijk[3] = {idx % n[0], (idx / n[0]) % n[1], idx / (n[0] * n[1])};
        int64_t off[3][3];                               /* off[a][0|1|2] = index offset of the -1 | 0 | +1 neighbour on axis a */
        int ok = 1;
        for (int a = 0; a < dim; ++a)
            for (int k = -1; k <= 1; ++k) {
                int64_t j = ijk[a] + k;
                if (j < 0 || j >= n[a]) { if (sper[a]) j = (j + n[a]) % n[a]; else ok = 0; }
                off[a][k + 1] = (j - ijk[a]) * stride[a];
            }
        double g[3], H[3][3], v[3][3];
        if (ok) {
#define S2(a, ka, b, kb) field[idx + off[a][(ka) + 1] + off[b][(kb) + 1]]
            double s0 = field[idx];
            ok = isfinite(s0);
            for (int a = 0; a < dim && ok; ++a) {
                double sp = field[idx + off[a][2]], sm = field[idx + off[a][0]];
                ok = isfinite(sp) && isfinite(sm);
                g[a] = (sp - sm) / (2.0 * dx[a]);
                H[a][a] = (sp - 2.0 * s0 + sm) / (dx[a] * dx[a]);
                for (int b = a + 1; b < dim && ok; ++b) {
                    double pp = S2(a, 1, b, 1), pm = S2(a, 1, b, -1), mp = S2(a, -1, b, 1), mm = S2(a, -1, b, -1);
                    ok = isfinite(pp) && isfinite(pm) && isfinite(mp) && isfinite(mm);
                    H[a][b] = H[b][a] = (pp - pm - mp + mm) / (4.0 * dx[a] * dx[b]);
                }
            }
#undef S2
        }
        if (!ok) { kappa[idx] = NAN; dgn[idx] = NAN; mask[idx] = 0; continue; }
        jacobi_sym(dim, H, v);
        int col = 0;
        for (int k = 1; k < dim; ++k) if (H[k][k] < H[col][col]) col = k;
        int big = 0;
        for (int r = 1; r < dim; ++r) if (fabs(v[r][col]) > fabs(v[big][col])) big = r;
        double sg = v[big][col] < 0.0 ? -1.0 : 1.0, d = 0.0;
        for (int r = 0; r < dim; ++r) d += g[r] * (sg * v[r][col]);
        double kap = H[col][col];
        kappa[idx] = kap;
        dgn[idx] = d;
        mask[idx] = (kap < -kappa_min && field[idx] >= s_min && fabs(d) <= fabs(kap) * delta / 2.0) ? 1 : 0;
    }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
