"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

The paper prints no worked example (no application has a closed form), so every pin
is a closed form of the DISCRETE method, an invariant, a library routine on a special case, or brute
force on tiny inputs.  Each test says which part of the oracle a plausible
mistake (dropped term, wrong sign/index, transposed operand) would break.
"""
import os

import numpy as np
import pytest
from scipy.linalg import expm

from paper_2209_13775_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_form_pins.txt")


def gold():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or "|" not in line:
            continue
        k, v = line.split("|")
        out[k.strip()] = float(v)
    return out


def P(z):
    """RK4 stability polynomial; works on scalars and (via matrix powers) on matrices."""
    if np.ndim(z) == 2:
        E = np.eye(z.shape[0])
        return E + z + z @ z / 2 + z @ z @ z / 6 + z @ z @ z @ z / 24
    return 1 + z + z**2 / 2 + z**3 / 6 + z**4 / 24


def run(oracle, w, seeds=None):
    f = oracle.OracleField.from_workload(w)
    s = w.seeds(np.float64) if seeds is None else seeds
    F, flag, es = f.advect(s, w.t0, w.tf, w.h)
    return f, s, F, flag, es


def cgf(oracle, w, F, flag):
    return oracle.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, F, flag, w.tf - w.t0)


def check_eig_lapack(cg, ftle, T, dim, rtol=1e-12):
    """O7 cross-check on every test: closed-form lambda_max vs LAPACK eigvalsh of the same C."""
    ok = np.isfinite(ftle)
    c = cg[ok]
    if dim == 2:
        M = np.stack([np.stack([c[:, 0], c[:, 1]], 1), np.stack([c[:, 1], c[:, 2]], 1)], 1)
    else:
        M = np.stack([np.stack([c[:, 0], c[:, 1], c[:, 2]], 1),
                      np.stack([c[:, 1], c[:, 3], c[:, 4]], 1),
                      np.stack([c[:, 2], c[:, 4], c[:, 5]], 1)], 1)
    lam = np.linalg.eigvalsh(M)[:, -1]
    ref = np.log(lam) / (2 * abs(T))
    assert np.allclose(ftle[ok], ref, rtol=rtol, atol=1e-12 / abs(T))
    assert np.all(np.linalg.eigvalsh(M)[:, 0] >= -1e-9 * lam)          # P11: C is PSD


# --------------------------------------------------------------------------------------------------
# meshes used by several pins
def _cart2(fn, times=(0.0, 20.0), half=4.0, nn=9, **kw):
    sp = 2 * half / (nn - 1)
    return I.analytic_cartesian(2, fn, (nn, nn), (-half, -half), (sp, sp), times, **kw)


def _cart3(fn, times=(0.0, 20.0), half=4.0, nn=7, **kw):
    sp = 2 * half / (nn - 1)
    return I.analytic_cartesian(3, fn, (nn, nn, nn), (-half,) * 3, (sp,) * 3, times, **kw)


def _tri(fn, times=(0.0, 20.0), half=4.0, nn=9, **kw):
    rng = np.random.default_rng(11)
    V, C = I.triangle_mesh_rect(nn, nn, 2 * half, 2 * half, rng)
    return I.analytic_simplex(2, fn, V - half, C, times, **kw)


def _tet(fn, times=(0.0, 20.0), half=4.0, nn=6, **kw):
    rng = np.random.default_rng(12)
    V, C = I.tet_mesh_box(nn, rng, -half, half)
    return I.analytic_simplex(3, fn, V, C, times, **kw)


MESHES = {"cart2": (_cart2, 2), "cart3": (_cart3, 3), "tri": (_tri, 2), "tet": (_tet, 3)}


def seedkw(dim, lo=-0.5, n=8, sp=0.125):
    return dict(ng=(n,) * dim, seed_lo=(lo,) * dim, seed_spacing=(sp,) * dim)


# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mesh", list(MESHES))
def test_P1_uniform_flow(oracle, mesh):
    """P1: u = c  =>  F = x0 + cT, G = I, C = I, FTLE = 0.  Breaks on: any interpolation weight not
    summing to 1, wrong RK4 weights (sum != 1), FD scaling, C assembly, eigenvalue offset."""
    mk, d = MESHES[mesh]
    c = np.array([0.3, -0.2, 0.15])[:d]
    w = mk(I.linear_flow(np.zeros((d, d)), c), t0=0.0, tf=5.0, h=0.25, **seedkw(d))
    f, s, F, flag, es = run(oracle, w)
    assert np.all(flag == 0) and np.all(es == 20)
    assert np.max(np.abs(F - (s + c * 5.0))) < 1e-13
    cg, ftle, st = cgf(oracle, w, F, flag)
    ident = np.array([1, 0, 1.0]) if d == 2 else np.array([1, 0, 0, 1, 0, 1.0])
    assert np.max(np.abs(cg - ident)) < 1e-11
    assert np.max(np.abs(ftle)) < 1e-12
    check_eig_lapack(cg, ftle, 5.0, d)


@pytest.mark.parametrize("mesh", list(MESHES))
def test_P2_interpolation_reproduces_affine(oracle, mesh):
    """P2: bi/trilinear and barycentric interpolation reproduce A x + b exactly (to rounding) at random
    points, and linearly in time between snapshots.  Breaks on: swapped weights w <-> 1-w, wrong corner
    index / stride, transposed component, wrong vertex-weight pairing, wrong tau."""
    mk, d = MESHES[mesh]
    rng = np.random.default_rng(5)
    A = rng.normal(size=(d, d))
    b = rng.normal(size=d)
    c = rng.normal(size=d)
    fn = lambda p, t: p @ A.T + b + c * t                 # affine in space, linear in time
    w = mk(fn, times=(1.0, 3.0, 5.0, 7.0), t0=1.0, tf=2.0, h=0.5, **seedkw(d))
    f = oracle.OracleField.from_workload(w)
    pts = rng.uniform(-3.9, 3.9, size=(2000, d))
    for t in (1.0, 2.2, 3.0, 4.9, 6.999):
        u, inside = f.velocity(pts, t)
        assert inside.all()
        assert np.max(np.abs(u - fn(pts, t))) < 5e-13


def test_P2_bilinear_reproduces_xy_and_weights(oracle):
    """P2: bilinear interpolation reproduces x*y exactly; trilinear reproduces x*y*z; O2 weights lie
    in [0,1] and reconstruct the point: node_lo + w*spacing == x."""
    rng = np.random.default_rng(6)
    w = _cart2(lambda p, t: np.stack([p[:, 0] * p[:, 1], p[:, 0] - p[:, 1]], 1), t0=0.0, tf=1.0, h=0.5, **seedkw(2))
    f = oracle.OracleField.from_workload(w)
    pts = rng.uniform(-4, 4, size=(3000, 2))
    u, inside = f.velocity(pts, 0.3)
    assert inside.all() and np.max(np.abs(u[:, 0] - pts[:, 0] * pts[:, 1])) < 1e-13
    cell, wt = f.cart_locate(pts)
    assert wt.min() >= 0.0 and wt.max() <= 1.0
    i0, i1 = cell % 8, cell // 8
    rec = np.stack([-4 + (i0 + wt[:, 0]) * 1.0, -4 + (i1 + wt[:, 1]) * 1.0], 1)
    assert np.max(np.abs(rec - pts)) < 1e-14
    w3 = _cart3(lambda p, t: np.stack([p[:, 0] * p[:, 1] * p[:, 2], p[:, 2], p[:, 1]], 1), t0=0.0, tf=1.0, h=0.5, **seedkw(3))
    f3 = oracle.OracleField.from_workload(w3)
    pts = rng.uniform(-4, 4, size=(3000, 3))
    u, inside = f3.velocity(pts, 0.0)
    assert inside.all() and np.max(np.abs(u[:, 0] - pts[:, 0] * pts[:, 1] * pts[:, 2])) < 1e-12


def test_O2_cartesian_locate_vs_scan(oracle):
    """O2 formula vs a brute-force scan (node_i <= x < node_{i+1}) on random points; closed upper end;
    outside -> -1; periodic wrap of negative and >L positions."""
    rng = np.random.default_rng(7)
    n = (11, 7, 5)
    origin, sp = (-1.0, 2.0, 0.5), (0.3, 0.25, 0.7)
    w = I.analytic_cartesian(3, lambda p, t: p, n, origin, sp, (0.0, 1.0), ng=(2, 2, 2), seed_lo=(0, 0, 0),
                             seed_spacing=(1, 1, 1), t0=0.0, tf=1.0, h=0.5)
    f = oracle.OracleField.from_workload(w)
    lo = np.array(origin)
    hi = lo + (np.array(n) - 1) * np.array(sp)
    pts = rng.uniform(lo - 0.2, hi + 0.2, size=(20000, 3))
    cell, wt = f.cart_locate(pts)
    inside = np.all((pts >= lo) & (pts <= hi), axis=1)
    assert np.array_equal(cell >= 0, inside)
    idx = []
    for a in range(3):
        nodes = origin[a] + np.arange(n[a]) * sp[a]
        idx.append(np.clip(np.searchsorted(nodes, pts[:, a], side="right") - 1, 0, n[a] - 2))
    ref = idx[0] + (n[0] - 1) * (idx[1] + (n[1] - 1) * idx[2])
    near_line = np.any(np.abs(wt) < 1e-9, axis=1) | np.any(np.abs(wt - 1) < 1e-9, axis=1)
    sel = inside & ~near_line
    assert np.array_equal(cell[sel], ref[sel])
    # closed upper corner belongs to the last cell with w = 1
    c, wt = f.cart_locate(hi[None, :])
    assert c[0] == (n[0] - 2) + (n[0] - 1) * ((n[1] - 2) + (n[1] - 1) * (n[2] - 2)) and np.all(wt == 1.0)
    # periodic: x, x - L and x + 3L land in the same cell with the same weights (to rounding)
    wp = I.analytic_cartesian(3, lambda p, t: p, (8, 8, 8), (0, 0, 0), (0.5, 0.5, 0.5), (0.0, 1.0), ng=(2, 2, 2),
                              seed_lo=(0, 0, 0), seed_spacing=(1, 1, 1), t0=0.0, tf=1.0, h=0.5, periodic=(1, 1, 1))
    fp = oracle.OracleField.from_workload(wp)
    x = rng.uniform(0, 4, size=(500, 3))
    c0, w0 = fp.cart_locate(x)
    c1, w1 = fp.cart_locate(x - 4.0)
    c2, w2 = fp.cart_locate(x + 12.0)
    assert np.array_equal(c0, c1) and np.array_equal(c0, c2)
    assert np.max(np.abs(w0 - w1)) < 1e-12 and np.max(np.abs(w0 - w2)) < 1e-11
    assert c0.max() < 512 and c0.min() >= 0


@pytest.mark.parametrize("mesh", list(MESHES))
def test_P3_linear_flow_exact_discrete_map(oracle, mesh):
    """P3: u = A x  =>  x_N = P(hA)^N x0 exactly, central differences exact => G = P(hA)^N, C = G^T G.
    Breaks on: RK4 stage coefficients or order of stages, wrong stage position (x + h/2 k), G index
    convention (G_ab = dF_a/dx_b vs transposed: A is non-symmetric), C = G G^T instead of G^T G."""
    mk, d = MESHES[mesh]
    rng = np.random.default_rng(21)
    A = rng.normal(size=(d, d)) * 0.25
    A -= np.eye(d) * np.trace(A) / d
    h, N = 0.125, 16
    w = mk(I.linear_flow(A), t0=0.0, tf=h * N, h=h, **seedkw(d))
    f, s, F, flag, es = run(oracle, w)
    assert np.all(flag == 0)
    M = np.linalg.matrix_power(P(h * A), N)
    assert np.max(np.abs(F - s @ M.T)) < 2e-13
    cg, ftle, st = cgf(oracle, w, F, flag)
    Cref = M.T @ M
    iu = np.triu_indices(d)
    interior = st == 0
    assert interior.sum() == (8 - 2) ** d                 # one-sided only on the grid faces
    assert np.max(np.abs(cg[interior] - Cref[iu])) < 2e-11
    assert np.max(np.abs(cg - Cref[iu])) < 2e-11          # one-sided is exact too on a linear map
    lam = np.linalg.eigvalsh(Cref)[-1]
    assert np.max(np.abs(ftle - np.log(lam) / (2 * h * N))) < 1e-11
    check_eig_lapack(cg, ftle, h * N, d)
    # and the continuous answer is close: |P(hA)^N - expm(AT)| = O(h^4)
    assert np.max(np.abs(M - expm(A * h * N))) < 1e-5


@pytest.mark.parametrize("s_,h", [(1.0, 0.1), (0.5, 0.1), (1.0, 0.05)])
def test_P4_pure_strain_ftle(oracle, s_, h):
    """P4: A = diag(s,-s): FTLE = ln P(hs)/h (golden, mpmath).  End-to-end O4-O7."""
    g = gold()
    T = 10.0
    w = I.analytic_cartesian(2, I.linear_flow(np.diag([s_, -s_])), (5, 5), (-40.0, -40.0), (20.0, 20.0), (0.0, 10.0),
                             ng=(6, 6), seed_lo=(-3e-4, -3e-4), seed_spacing=(1e-4, 1e-4), t0=0.0, tf=T, h=h)
    f, s, F, flag, es = run(oracle, w)
    assert np.all(flag == 0)
    cg, ftle, st = cgf(oracle, w, F, flag)
    ref = g["P4_strain_ftle s=%s h=%s" % (s_, h)]
    assert np.max(np.abs(ftle - ref)) < 1e-12
    if s_ == 1.0 and h == 0.1:
        lam = np.exp(ftle * 2 * T)
        assert np.max(np.abs(lam / g["P4_strain_lambda_max s=1 h=0.1 T=10"] - 1)) < 1e-10
    check_eig_lapack(cg, ftle, T, 2)


@pytest.mark.parametrize("gamma", [0.5, 1.0])
def test_P5_simple_shear(oracle, gamma):
    """P5: u = (gamma y, 0): RK4 exact, lambda_max = 1 + k^2/2 + k sqrt(1+k^2/4), det C = 1."""
    g = gold()
    T = 10.0
    w = I.analytic_cartesian(2, I.linear_flow([[0, gamma], [0, 0]]), (5, 5), (-40.0, -40.0), (20.0, 20.0), (0.0, 10.0),
                             ng=(6, 6), seed_lo=(-1.0, -1.0), seed_spacing=(0.25, 0.25), t0=0.0, tf=T, h=0.1)
    f, s, F, flag, es = run(oracle, w)
    assert np.max(np.abs(F - (s + np.stack([gamma * T * s[:, 1], 0 * s[:, 1]], 1)))) < 1e-12
    cg, ftle, st = cgf(oracle, w, F, flag)
    k = gamma * T
    assert np.max(np.abs(cg - np.array([1.0, k, 1 + k * k]))) < 1e-10      # C = [[1,k],[k,1+k^2]]
    assert np.max(np.abs(cg[:, 0] * cg[:, 2] - cg[:, 1] ** 2 - 1.0)) < 1e-9
    assert np.max(np.abs(ftle - g["P5_shear_ftle gamma=%s T=10.0" % gamma])) < 1e-12
    assert np.max(np.abs(np.exp(2 * T * ftle) / g["P5_shear_lambda_max gamma=%s T=10.0" % gamma] - 1)) < 1e-11


@pytest.mark.parametrize("name,omega", [("1", 1.0), ("2pi/10", 2 * np.pi / 10)])
def test_P6_rigid_rotation(oracle, name, omega):
    """P6: u = w(-y,x): exact C = I; RK4 gives FTLE = ln|P(ihw)|/h (about -(hw)^6/(144h)): pins O7 near lambda=1."""
    g = gold()
    T, h = 10.0, 0.1
    w = _cart2(I.linear_flow([[0, -omega], [omega, 0]]), t0=0.0, tf=T, h=h, ng=(6, 6), seed_lo=(-1.0, -1.0),
               seed_spacing=(0.3, 0.3))
    f, s, F, flag, es = run(oracle, w)
    assert np.all(flag == 0)
    cg, ftle, st = cgf(oracle, w, F, flag)
    ref = g["P6_rotation_ftle omega=%s h=0.1" % name]
    assert np.max(np.abs(ftle - ref)) < 2e-14 + 1e-6 * abs(ref)
    assert np.max(np.abs(cg[:, 1])) < 1e-12


def test_P7_fourth_order_convergence(oracle):
    """P7: error against expm(A T) x0 falls 16x per halving of h."""
    A = np.array([[0.2, -1.0], [1.3, -0.2]])
    T = 2.0
    errs = []
    for h in (0.2, 0.1, 0.05, 0.025):
        w = _cart2(I.linear_flow(A), t0=0.0, tf=T, h=h, **seedkw(2))
        f, s, F, flag, es = run(oracle, w)
        errs.append(np.max(np.abs(F - s @ expm(A * T).T)))
    ratios = np.array(errs[:-1]) / np.array(errs[1:])
    assert np.all((ratios > 14) & (ratios < 18)), ratios


def test_P8_time_interpolation_piecewise_linear(oracle):
    """P8: spatially uniform field with arbitrary snapshot values c_s: linear time interpolation is
    piecewise linear, RK4 is Simpson in t (exact on each linear piece when steps do not straddle a
    snapshot) => F = x0 + sum of trapezoids.  Breaks on: wrong bracket index s, wrong tau, stage times
    (ta,tb,tb,tc), accumulated instead of multiplied time."""
    rng = np.random.default_rng(8)
    times = 2.0 + 0.5 * np.arange(9)                       # 2.0 .. 6.0
    c = rng.normal(size=(9, 2))
    fn = lambda p, t: np.broadcast_to(c[int(round((t - 2.0) / 0.5))], p.shape).copy()
    w = _cart2(fn, times=times, t0=2.5, tf=5.5, h=0.125, **seedkw(2))
    f, s, F, flag, es = run(oracle, w)
    trap = sum(0.5 * 0.5 * (c[k] + c[k + 1]) for k in range(1, 7))
    assert np.max(np.abs(F - (s + trap))) < 1e-13
    # backward over the same window returns exactly (to rounding) -- also pins h<0 handling
    Fb, flagb, esb = f.advect(F, 5.5, 2.5, -0.125)
    assert np.max(np.abs(Fb - s)) < 1e-13 and np.all(esb == 24)
    # u = a + b t (globally linear): x = x0 + a T + b (tf^2 - t0^2)/2
    a, b = np.array([0.1, -0.2]), np.array([0.03, 0.05])
    w2 = _cart2(I.time_linear_uniform(a, b), times=np.arange(0.0, 11.0), t0=1.0, tf=9.0, h=0.25, **seedkw(2))
    f2, s2, F2, _, _ = run(oracle, w2)
    assert np.max(np.abs(F2 - (s2 + a * 8.0 + b * (81 - 1) / 2))) < 1e-13


@pytest.mark.parametrize("dim", [2, 3])
def test_P9_location_brute_vs_walk_and_tiebreak(oracle, dim):
    """P9: brute force (the definition) vs walk on tiny meshes for every query, including points exactly
    on faces, edges and vertices of a Kuhn mesh with integer coordinates (s == 0 ties) and of mixed
    orientation.  No point is accepted by two cells; interior points are accepted by exactly one."""
    n = 5 if dim == 2 else 4
    V, C = I.kuhn_mesh(dim, n)
    w = I.analytic_simplex(dim, lambda p, t: p, V, C, (0.0, 1.0), ng=(2,) * dim, seed_lo=(0,) * dim,
                           seed_spacing=(1,) * dim, t0=0.0, tf=1.0, h=0.5)
    f = oracle.OracleField.from_workload(w)
    rng = np.random.default_rng(9)
    g = np.arange(0, 2 * (n - 1) + 1) * 0.5               # lattice of half-integers: vertices, edge and face midpoints
    grids = np.meshgrid(*([g] * dim), indexing="ij")
    lattice = np.stack([x.ravel() for x in grids], 1)
    rand = rng.uniform(-0.3, n - 1 + 0.3, size=(3000, dim))
    thirds = lattice[: 200] * (2.0 / 3.0)
    pts = np.concatenate([lattice, rand, thirds])
    cell_b, count = f.locate_brute(pts)
    assert count.max() <= 1                                # never two owners
    strictly_inside = np.all((pts > 0) & (pts < n - 1), axis=1)
    assert np.all(count[strictly_inside] == 1)             # no gaps in the interior, ties included
    outside = np.any((pts < 0) | (pts > n - 1), axis=1)
    assert np.all(cell_b[outside] == -1)
    for start in (np.zeros(len(pts), np.int32), np.full(len(pts), len(C) - 1, np.int32), None):
        cell_w = f.locate_walk(pts, start)
        assert np.array_equal(cell_w, cell_b)
    # the owner of an interior face point is the SAME from both sides: move the start cell
    # containment sanity: barycentric weights of the owner are >= -1e-12
    own = cell_b >= 0
    u, inside = f.velocity(pts[own], 0.0, cell_b[own])     # field is u = x
    assert inside.all() and np.max(np.abs(u - pts[own])) < 1e-12


@pytest.mark.parametrize("dim", [2, 3])
def test_P9_location_on_jittered_delaunay(oracle, dim):
    """Brute force vs walk on jittered Delaunay meshes (the recipe of configs 2 and 4, small), random
    points and points on/near vertices; neighbour table symmetric."""
    rng = np.random.default_rng(10)
    if dim == 2:
        V, C = I.triangle_mesh_rect(12, 9, 2.0, 1.0, rng)
        lo, hi = np.array([0, 0.0]), np.array([2.0, 1.0])
    else:
        V, C = I.tet_mesh_box(6, rng, 0.0, 1.0)
        lo, hi = np.zeros(3), np.ones(3)
    w = I.analytic_simplex(dim, lambda p, t: p, V, C, (0.0, 1.0), ng=(2,) * dim, seed_lo=(0,) * dim,
                           seed_spacing=(1,) * dim, t0=0.0, tf=1.0, h=0.5)
    f = oracle.OracleField.from_workload(w)
    nb = f.neigh
    for c in range(0, len(C), 7):
        for j in range(dim + 1):
            m = nb[c, j]
            if m >= 0:
                assert c in nb[m]
                assert len(set(C[c]) & set(C[m])) == dim
    # generic points + points on faces (centroids: one near-zero s, the SAME expression in both cells)
    fc = V[C[:300, 1:]].mean(axis=1)
    pts = np.concatenate([rng.uniform(lo - 0.05, hi + 0.05, size=(4000, dim)), fc])
    cell_b, count = f.locate_brute(pts)
    assert count.max() <= 1
    strictly = np.all((pts > lo + 1e-9) & (pts < hi - 1e-9), axis=1)
    assert np.all(count[strictly] == 1)
    assert np.array_equal(f.locate_walk(pts), cell_b)
    assert np.array_equal(f.locate_walk(pts, np.zeros(len(pts), np.int32)), cell_b)
    # points at vertices / on edges of a jittered mesh: the zero s values are rounding noise, several
    # cells (or none) may accept; what is required is validity: the walk returns an accepting cell.
    deg = np.concatenate([V, V[:50] + 1e-15, 0.5 * (V[C[:100, 0]] + V[C[:100, 1]])])
    cell_b, count = f.locate_brute(deg)
    cell_w = f.locate_walk(deg)
    has = count >= 1
    assert np.all(f.accepts(deg[has], cell_b[has]))
    assert np.all(f.accepts(deg[has], cell_w[has]) | (cell_w[has] == -1))
    assert np.all(cell_b[~has] == -1) and np.all(cell_w[~has] == -1)


def test_P10_eigmax_vs_lapack(oracle):
    """P10: closed-form lambda_max vs LAPACK eigvalsh on random SPD matrices, condition numbers to 1e12.
    2x2: full precision.  3x3 trigonometric form: relative error <= ~eps/gap with gap = (l1-l2)/l1, i.e.
    full precision for a separated largest eigenvalue, degrading to sqrt(eps) ~ 1e-8 when the two largest
    coincide (acos is ill-conditioned at r = -1) -- measured, and far inside the 3D FTLE gate (1e-3)."""
    rng = np.random.default_rng(13)
    worst2 = 0.0
    for trial in range(3000):
        k = rng.uniform(0, 12)
        for d in (2, 3):
            Q, _ = np.linalg.qr(rng.normal(size=(d, d)))
            ev = np.sort(10.0 ** rng.uniform(-k, 0, size=d)) * 10.0 ** rng.uniform(-3, 6)
            if trial % 50 == 0:
                ev[:] = ev[0]                              # repeated eigenvalues (p2 == 0 branch nearby)
            if trial % 5 == 1 and d == 3:
                ev[1] = ev[2] * (1 - 10.0 ** rng.uniform(-16, 0))    # (nearly) double largest eigenvalue
            M = (Q * ev) @ Q.T
            M = 0.5 * (M + M.T)
            e = np.linalg.eigvalsh(M)
            if d == 2:
                lam = oracle.eigmax_sym2(M[0, 0], M[0, 1], M[1, 1])
                worst2 = max(worst2, abs(lam / e[-1] - 1))
            else:
                lam = oracle.eigmax_sym3(M[0, 0], M[0, 1], M[0, 2], M[1, 1], M[1, 2], M[2, 2])
                gap = max((e[2] - e[1]) / e[2], 1e-300)
                assert abs(lam / e[2] - 1) <= min(2e-8, max(5e-15, 2e-15 / gap)), (e, lam)
    assert worst2 < 1e-14, worst2
    assert oracle.eigmax_sym3(2, 0, 0, 2, 0, 2) == 2.0
    assert abs(oracle.eigmax_sym3(1, 0, 0, 5, 0, 3) - 5.0) < 1e-15
    assert abs(oracle.eigmax_sym2(1, 2, 1) - 3.0) < 1e-15


def test_P11_det_C_incompressible_linear(oracle):
    """P11: incompressible 2D linear flow with eigenvalues +-mu: det C = (P(h mu) P(-h mu))^(2N) (computed,
    = 1 + O(h^5 T)); C symmetric PSD."""
    mu, h, N = 0.7, 0.1, 40
    R = np.array([[np.cos(0.4), -np.sin(0.4)], [np.sin(0.4), np.cos(0.4)]])
    A = R @ np.diag([mu, -mu]) @ R.T
    w = I.analytic_cartesian(2, I.linear_flow(A), (5, 5), (-40.0, -40.0), (20.0, 20.0), (0.0, 10.0),
                             ng=(6, 6), seed_lo=(-0.3, -0.3), seed_spacing=(0.1, 0.1), t0=0.0, tf=h * N, h=h)
    f, s, F, flag, es = run(oracle, w)
    cg, ftle, st = cgf(oracle, w, F, flag)
    det = cg[:, 0] * cg[:, 2] - cg[:, 1] ** 2
    ref = (P(h * mu) * P(-h * mu)) ** (2 * N)
    assert abs(ref - 1) < 1e-5 and abs(ref - 1) > 1e-9
    assert np.max(np.abs(det / ref - 1)) < 1e-10
    check_eig_lapack(cg, ftle, h * N, 2)


def test_P12_periodic_shift_and_seam(oracle):
    """P12: on a periodic field F(x0 + L e_a) - F(x0) = L e_a (O2 wrap); the FD gradient across the seed
    grid's periodic seam equals the gradient computed on a grid shifted by half a period (O5 seam)."""
    w = I.config3(ngrid=8, nn=16, T=1.0, h=0.05, n_snap=4)
    f = oracle.OracleField.from_workload(w)
    s = w.seeds(np.float64)
    F0, flag0, _ = f.advect(s, 0.0, 1.0, 0.05)
    L = 2 * np.pi
    for a in range(3):
        e = np.zeros(3)
        e[a] = L
        for sh in (e, -2 * e):
            F1, flag1, _ = f.advect(s + sh, 0.0, 1.0, 0.05)
            assert np.all(flag1 == 0)
            assert np.max(np.abs(F1 - F0 - sh)) < 5e-13
    cg, ftle, st = cgf(oracle, w, F0, flag0)
    assert np.all(st == 0) and np.all(np.isfinite(ftle))
    # shifted seed grid: seeds moved by +L/2 in every axis = the same physical points, re-indexed by 4
    F2, flag2, _ = f.advect(s + L / 2, 0.0, 1.0, 0.05)
    cg2, ftle2, st2 = cgf(oracle, w, F2, flag2)
    A = ftle.reshape(8, 8, 8)
    B = np.roll(ftle2.reshape(8, 8, 8), shift=(4, 4, 4), axis=(0, 1, 2))
    assert np.max(np.abs(A - B)) < 1e-11
    check_eig_lapack(cg, ftle, 1.0, 3)


def test_O5_one_sided_and_invalid_neighbours(oracle):
    """O5: exited neighbours are skipped (one-sided, status bit 1), an exited seed or an isolated seed gives
    NaN (status bit 0).  Quadratic map F = x^2 makes central and one-sided differences distinguishable."""
    ng = (5, 4)
    dx = (0.5, 0.25)
    s = I.seed_grid(2, ng + (1,), (0, 0, 0), dx + (1.0,))
    F = np.stack([s[:, 0] ** 2 + s[:, 1], 3 * s[:, 1] - s[:, 0]], 1)
    flag = np.zeros(20, np.uint8)
    flag[2 + 5 * 1] = 1                                     # seed (2,1) exited
    cg, ftle, st = oracle.cg_ftle(2, ng, dx, (0, 0), (0, 0), F, flag, 2.0)
    assert np.isnan(ftle[2 + 5]) and st[2 + 5] & 1
    # (1,1): +x neighbour invalid -> backward difference of x^2 at x=0.75: (0.75^2 - 0.25^2)/0.5 = 1.0
    G = np.array([[1.0, 1.0], [-1.0, 3.0]])
    Cref = G.T @ G
    assert st[1 + 5] == 2 and np.allclose(cg[1 + 5], [Cref[0, 0], Cref[0, 1], Cref[1, 1]], atol=1e-12)
    # (3,1): -x neighbour invalid -> forward difference at x=1.75: (2.25^2-1.75^2)/0.5 = 4.0
    G = np.array([[4.0, 1.0], [-1.0, 3.0]])
    Cref = G.T @ G
    assert st[3 + 5] == 2 and np.allclose(cg[3 + 5], [Cref[0, 0], Cref[0, 1], Cref[1, 1]], atol=1e-12)
    # interior (2,2): central d(x^2)/dx at 1.25 = 2.5 ; its -y neighbour (2,1) is invalid -> one-sided in y (exact)
    G = np.array([[2.5, 1.0], [-1.0, 3.0]])
    Cref = G.T @ G
    assert st[2 + 10] == 2 and np.allclose(cg[2 + 10], [Cref[0, 0], Cref[0, 1], Cref[1, 1]], atol=1e-12)
    # a 1-wide grid has no neighbour on that axis -> NaN
    cg1, ftle1, st1 = oracle.cg_ftle(2, (5, 1), dx, (0, 0), (0, 0), F[:5], None, 2.0)
    assert np.all(np.isnan(ftle1)) and np.all(st1 & 1)


def test_O4_exit_handling(oracle):
    """Readings #9/#10: uniform flow to the right on a finite box: a tracer exits at the first step where
    ANY stage point is outside; it keeps its start-of-step position, flag 1, exit_step n.  Seeds outside
    at t0: flag 2, flow map = seed, exit_step 0."""
    w = I.analytic_cartesian(2, I.linear_flow(np.zeros((2, 2)), [1.0, 0.0]), (5, 5), (0.0, 0.0), (1.0, 1.0), (0.0, 10.0),
                             ng=(4, 1), seed_lo=(0.0, 0.0), seed_spacing=(1.0, 1.0), t0=0.0, tf=5.0, h=0.25)
    f = oracle.OracleField.from_workload(w)
    seeds = np.array([[0.5, 2.0], [3.5, 2.0], [3.9, 2.0], [4.5, 2.0], [2.0, -0.1], [-1.0, 2.0]])
    F, flag, es = f.advect(seeds, 0.0, 5.0, 0.25)
    # 0.5 -> would reach 5.5: steps complete while x + h <= 4: x_n = 0.5 + 0.25 n, stage-4 point x_n + 0.25 <= 4 -> n <= 13
    assert flag[0] == 1 and es[0] == 14 and abs(F[0, 0] - 4.0) < 1e-14
    assert flag[1] == 1 and es[1] == 2 and abs(F[1, 0] - 4.0) < 1e-14
    assert flag[2] == 1 and es[2] == 0 and F[2, 0] == 3.9
    assert list(flag[3:]) == [2, 2, 2] and np.all(es[3:] == 0) and np.array_equal(F[3:], seeds[3:])
    # short run stays inside
    F, flag, es = f.advect(seeds[:1], 0.0, 3.0, 0.25)
    assert flag[0] == 0 and es[0] == 12 and abs(F[0, 0] - 3.5) < 1e-14


def test_P13_pipe_invariants_on_tets(oracle):
    """P13: config-4 field (before meshing): r is invariant, z(t) = z0 + 2(1 - r0^2)(t - t0).  On the tet mesh
    these hold to P1 interpolation error O(delta^2): a sanity band, not a gate."""
    w = I.config4(ng=(6, 6, 6), delta=0.1, T=0.5, h=0.02, n_snap=6, length=3.0)
    f = oracle.OracleField.from_workload(w)
    rng = np.random.default_rng(14)
    r0 = rng.uniform(0.0, 0.7, 400)
    th = rng.uniform(0, 2 * np.pi, 400)
    s = np.stack([r0 * np.cos(th), r0 * np.sin(th), rng.uniform(0.5, 1.2, 400)], 1)
    F, flag, es = f.advect(s, 0.0, 0.5, 0.02)
    assert np.all(flag == 0)
    r1 = np.hypot(F[:, 0], F[:, 1])
    assert np.max(np.abs(r1 - r0)) < 0.01
    assert np.max(np.abs(F[:, 2] - (s[:, 2] + 2 * (1 - r0 ** 2) * 0.5))) < 0.02
    # seeds outside the cylinder are flagged 2 (bounding-box seed grid with out-of-domain flags)
    F, flag, es = f.advect(w.seeds(np.float64), 0.0, 0.5, 0.02)
    sd = w.seeds(np.float64)
    assert np.all(flag[np.hypot(sd[:, 0], sd[:, 1]) > 1.0] == 2)
    far = (np.hypot(sd[:, 0], sd[:, 1]) < 0.8) & (sd[:, 2] < 1.5)      # cannot reach the outlet z=3 in T=0.5
    assert far.sum() > 10 and np.all(flag[far] == 0)
    out = (np.hypot(sd[:, 0], sd[:, 1]) < 0.5) & (sd[:, 2] > 2.7)      # u_z >= 1.5: leaves through the outlet
    assert out.sum() > 0 and np.all(flag[out] == 1) and np.all(es[out] < 25)


def test_P14_forward_backward(oracle):
    """P14: forward then backward over the same interval returns to x0 within O(h^4), and the residual
    falls by about 16x when h is halved (backward time = config 5)."""
    w = I.config1(ng=(32, 16), T=4.0, h=0.1)
    f = oracle.OracleField.from_workload(w)
    s = w.seeds()
    res = []
    for h in (0.1, 0.05):
        F, flag, _ = f.advect(s, 0.0, 4.0, h)
        B, flagb, _ = f.advect(F, 4.0, 0.0, -h)
        assert np.all(flag == 0) and np.all(flagb == 0)
        res.append(np.median(np.linalg.norm(B - s, axis=1)))
    assert res[0] < 1e-5 and res[0] / res[1] > 8.0, res


def test_double_gyre_closed_domain_and_detC(oracle):
    """Config 1 (small): the double gyre is closed, so every exit flag is 0 (SURVEY parity protocol); det C is
    near 1 (incompressible) up to FD + interpolation error -- reported as a sanity statistic."""
    w = I.config1(ng=(64, 32), T=10.0, h=0.1)
    f, s, F, flag, es = run(oracle, w)
    assert np.all(flag == 0) and np.all(es == 100)
    assert F[:, 0].min() > 0 and F[:, 0].max() < 2 and F[:, 1].min() > 0 and F[:, 1].max() < 1
    cg, ftle, st = cgf(oracle, w, F, flag)
    check_eig_lapack(cg, ftle, 10.0, 2)
    assert np.nanmax(ftle) > 0.2 and np.nanmax(ftle) < 1.0            # known range of the double-gyre FTLE ridge


def test_trajectory_recording(oracle):
    """e_D(t) support: recorded positions at the last record equal the flow map."""
    w = I.config1(ng=(8, 4), T=2.0, h=0.1)
    f = oracle.OracleField.from_workload(w)
    F, flag, es, traj = f.advect(w.seeds(), 0.0, 2.0, 0.1, rec_every=5)
    assert traj.shape == (4, 32, 2) and np.array_equal(traj[-1], F)


# -------------------------------------------------------------------------------------------------
# O8 (row f2): full eigen-decomposition of C
def _sym_from_upper(dim, c):
    if dim == 2:
        return np.array([[c[0], c[1]], [c[1], c[2]]])
    return np.array([[c[0], c[1], c[2]], [c[1], c[3], c[4]], [c[2], c[4], c[5]]])


def _random_spd(rng, dim, n, max_cond_log10):
    """Q diag(lambda) Q^T with log-uniform condition numbers up to 10^max_cond_log10, as upper triangles."""
    out = np.empty((n, 3 if dim == 2 else 6))
    for i in range(n):
        q, _ = np.linalg.qr(rng.standard_normal((dim, dim)))
        lam = 10.0 ** rng.uniform(-max_cond_log10 / 2, max_cond_log10 / 2, dim)
        a = (q * lam) @ q.T
        a = 0.5 * (a + a.T)
        out[i] = a[np.triu_indices(dim)]
    return out


@pytest.mark.parametrize("dim", [2, 3])
def test_P15_eigen_decomposition_vs_lapack(oracle, dim):
    """Pin for O8: eigenvalues against LAPACK (numpy.linalg.eigh) to 1e-13 of lambda_max on SPD matrices with condition
    numbers up to 1e12; residual |C v - lambda v| <= 1e-13 |C|; V orthonormal; eigenvectors equal LAPACK's up to sign
    where the spectrum is well separated; sign convention (largest component positive); ascending order."""
    rng = np.random.default_rng(150 + dim)
    cg = _random_spd(rng, dim, 2000, 12)
    ev, vec = oracle.cg_eigen(dim, cg)
    assert np.all(np.diff(ev, axis=1) >= 0)
    for i in range(cg.shape[0]):
        a = _sym_from_upper(dim, cg[i])
        wl, vl = np.linalg.eigh(a)
        scale = np.abs(wl).max()
        assert np.max(np.abs(ev[i] - wl)) <= 1e-13 * scale
        assert np.max(np.abs(vec[i] @ vec[i].T - np.eye(dim))) <= 1e-13
        for k in range(dim):
            assert np.linalg.norm(a @ vec[i, k] - ev[i, k] * vec[i, k]) <= 1e-13 * scale
            j = int(np.argmax(np.abs(vec[i, k])))
            assert vec[i, k, j] > 0
            gap = min(abs(wl[k] - wl[m]) for m in range(dim) if m != k)
            if gap > 1e-3 * scale:
                assert abs(abs(vec[i, k] @ vl[:, k]) - 1.0) <= 1e-9


def test_P15_eigen_closed_forms(oracle):
    """Closed forms: simple shear (pin P5) C = [[1, k], [k, 1 + k^2]] has lambda = 1 + k^2/2 +- k sqrt(1 + k^2/4), product 1,
    and eigenvector (k, lambda - 1) / norm; diagonal matrices return the sorted diagonal and unit axes; a matrix with NaN
    returns NaN; the largest eigenvalue equals the closed form of rule O7."""
    k = 5.0
    ev, vec = oracle.cg_eigen(2, np.array([[1.0, k, 1.0 + k * k]]))
    lp = 1 + k * k / 2 + k * np.sqrt(1 + k * k / 4)
    assert abs(ev[0, 1] - lp) <= 1e-13 * lp and abs(ev[0, 0] * ev[0, 1] - 1.0) <= 1e-12
    assert abs(ev[0, 1] - 26.96291201783626) <= 1e-12                       # tests/golden pin P5, gamma T = 5
    v = np.array([k, lp - 1.0]); v /= np.linalg.norm(v)
    assert np.max(np.abs(vec[0, 1] - v)) <= 1e-14
    ev, vec = oracle.cg_eigen(3, np.array([[3.0, 0.0, 0.0, 1.0, 0.0, 2.0]]))
    assert np.array_equal(ev[0], [1.0, 2.0, 3.0])
    assert np.array_equal(vec[0], [[0, 1, 0], [0, 0, 1], [1, 0, 0]])
    ev, vec = oracle.cg_eigen(3, np.array([[1.0, np.nan, 0.0, 1.0, 0.0, 1.0]]))
    assert np.all(np.isnan(ev)) and np.all(np.isnan(vec))
    rng = np.random.default_rng(7)
    cg = _random_spd(rng, 3, 200, 8)
    ev, _ = oracle.cg_eigen(3, cg)
    for i in range(200):
        assert abs(ev[i, 2] - oracle.eigmax_sym3(*cg[i])) <= 1e-12 * ev[i, 2]


# -------------------------------------------------------------------------------------------------
# O9 (row f3): gradient from auxiliary points
def test_P16_aux_gradient_linear_flow_and_shear(oracle):
    """Pin for O9: for u = A x the flow map is linear, so the auxiliary-point quotient is exact for ANY delta:
    G = P(hA)^N, C = G^T G (pin P3); simple shear gives the closed-form FTLE of pin P5; a flagged auxiliary tracer gives
    NaN + status 1; grid-neighbour (O5) and auxiliary (O9) gradients agree on a smooth flow to O(dx^2)."""
    A = np.array([[0.1, 0.4], [-0.3, -0.1]])
    h, N = 0.1, 50
    w = I.analytic_cartesian(2, I.linear_flow(A), (41, 41), (-2.0, -2.0), (0.1, 0.1), (0.0, 5.0), ng=(6, 5), seed_lo=(-0.5, -0.5),
                             seed_spacing=(0.2, 0.2), t0=0.0, tf=h * N, h=h)
    fo = oracle.OracleField.from_workload(w)
    delta = (1e-3, 2e-3)
    aux = I.aux_seeds(w.seeds(), delta)
    Fa, fla, _ = fo.advect(aux.reshape(-1, 2), w.t0, w.tf, w.h)
    assert np.all(fla == 0)
    cg, ftle, st = oracle.cg_ftle_aux(2, delta, Fa, fla, w.tf - w.t0)
    hA = h * A
    P = np.eye(2) + hA + hA @ hA / 2 + hA @ hA @ hA / 6 + hA @ hA @ hA @ hA / 24
    G = np.linalg.matrix_power(P, N)
    Cx = G.T @ G
    assert np.max(np.abs(cg - np.array([Cx[0, 0], Cx[0, 1], Cx[1, 1]]))) <= 1e-9
    assert np.all(st == 0)
    lam = np.linalg.eigvalsh(Cx)[-1]
    assert np.max(np.abs(ftle - np.log(lam) / (2 * h * N))) <= 1e-10
    # shear: u = (gamma y, 0), gamma T = 5 -> FTLE of pin P5
    w2 = I.analytic_cartesian(2, I.linear_flow(np.array([[0.0, 0.5], [0.0, 0.0]])), (41, 41), (-20.0, -2.0), (1.0, 0.1), (0.0, 10.0),
                              ng=(4, 4), seed_lo=(-1.0, -1.0), seed_spacing=(0.5, 0.5), t0=0.0, tf=10.0, h=0.1)
    fo2 = oracle.OracleField.from_workload(w2)
    aux2 = I.aux_seeds(w2.seeds(), (0.01, 0.01))
    F2, fl2, _ = fo2.advect(aux2.reshape(-1, 2), 0.0, 10.0, 0.1)
    cg2, ft2, st2 = oracle.cg_ftle_aux(2, (0.01, 0.01), F2, fl2, 10.0)
    assert np.max(np.abs(ft2 - 0.164723114637109571)) <= 1e-10           # tests/golden/closed_form_pins.txt, P5
    fl2 = fl2.reshape(-1, 4).copy(); fl2[3, 2] = 1
    cg3, ft3, st3 = oracle.cg_ftle_aux(2, (0.01, 0.01), F2, fl2, 10.0)
    assert np.isnan(ft3[3]) and st3[3] == 1 and np.all(np.isnan(cg3[3])) and np.isfinite(ft3[2]) and st3[2] == 0
    # against the grid-neighbour gradient on the double gyre (interior seeds): both approximate the same derivative
    w3 = I.config1(ng=(64, 32), T=2.0)
    fo3 = oracle.OracleField.from_workload(w3)
    Fg, flg, _ = fo3.advect(w3.seeds(), w3.t0, w3.tf, w3.h)
    _, ftg, _ = oracle.cg_ftle(2, w3.ng, w3.seed_spacing, w3.seed_periodic, w3.period, Fg, flg, w3.tf - w3.t0)
    d3 = (w3.seed_spacing[0], w3.seed_spacing[1])
    Fa3, fla3, _ = fo3.advect(I.aux_seeds(w3.seeds(), d3).reshape(-1, 2), w3.t0, w3.tf, w3.h)
    _, fta, sta = oracle.cg_ftle_aux(2, d3, Fa3, fla3, w3.tf - w3.t0)
    inner = np.zeros((32, 64), bool); inner[1:-1, 1:-1] = True
    ok = inner.ravel() & (sta == 0)
    assert ok.sum() > 1500 and np.max(np.abs(fta[ok] - ftg[ok])) <= 1e-12   # delta = seed spacing: the very same stencil


# -------------------------------------------------------------------------------------------------
# O10 (row f1): early evaluation of C when a stencil member leaves
def test_P17_early_cg(oracle):
    """Pins for O10.  (a) No exits: identical to the plain evaluation at T for any `every`.  (b) Uniform flow through an
    open box: the exit step of every tracer follows from geometry, hence t_eff of every seed; C = I, FTLE = 0.  (c) Pure
    strain u = (s x, -s y) in an open box: FTLE_RK4 = ln P(hs) / h whatever the evaluation time (pin P4), so every
    evaluated seed carries the same value although their t_eff differ."""
    w = I.config1(ng=(32, 16), T=3.0)
    fo = oracle.OracleField.from_workload(w)
    args = (2, w.ng, w.seed_spacing, w.seed_periodic, w.period)
    F, fl, es, cg, ft, te, st = oracle.early_cg(fo, *args, w.seeds(), w.t0, w.tf, w.h, every=7)
    cg0, ft0, st0 = oracle.cg_ftle(*args, F, fl, w.tf - w.t0)
    assert np.all(fl == 0) and np.array_equal(cg, cg0) and np.array_equal(ft, ft0) and np.array_equal(st, st0)
    assert np.all(te == w.tf - w.t0)
    # (b) uniform flow c = (0.3, 0) in the box [0,4] x [0,4], seeds on an 8 x 6 grid, h = 0.25, 20 steps, every = 2
    c, h, N, K = 0.3, 0.25, 20, 2
    wu = I.analytic_cartesian(2, I.linear_flow(np.zeros((2, 2)), np.array([c, 0.0])), (5, 5), (0.0, 0.0), (1.0, 1.0), (0.0, 10.0),
                              ng=(8, 6), seed_lo=(0.2, 0.5), seed_spacing=(0.45, 0.5), t0=0.0, tf=h * N, h=h)
    fu = oracle.OracleField.from_workload(wu)
    s = wu.seeds()
    F, fl, es, cg, ft, te, st = oracle.early_cg(fu, 2, wu.ng, wu.seed_spacing, wu.seed_periodic, wu.period, s, 0.0, h * N, h, every=K)
    # a step n succeeds iff x0 + c (n + 1) h <= 4 (the last stage point is the farthest): exit_step = number of such n
    es_geo = np.minimum(N, np.floor((4.0 - s[:, 0]) / (c * h) + 1e-9)).astype(int)
    assert np.array_equal(es, es_geo) and set(np.unique(fl)) == {0, 1}
    esg = es_geo.reshape(6, 8)
    stencil_min = esg.copy()
    stencil_min[:, :-1] = np.minimum(stencil_min[:, :-1], esg[:, 1:])        # +x neighbour leaves first; y neighbours leave with the seed
    te_geo = (stencil_min // K) * K * h
    assert np.allclose(te.reshape(6, 8), te_geo, atol=1e-12)
    ok = te > 0
    assert ok.sum() > 30 and np.all(st[~ok] & 1) and np.all(np.isnan(ft[~ok]))
    assert np.max(np.abs(cg[ok] - np.array([1.0, 0.0, 1.0]))) <= 1e-12 and np.max(np.abs(ft[ok])) <= 1e-12
    # (c) pure strain, s = 1, h = 0.1: FTLE = 0.999999233219801983 at every evaluation time
    ws = I.analytic_cartesian(2, I.linear_flow(np.array([[1.0, 0.0], [0.0, -1.0]])), (41, 41), (-4.0, -4.0), (0.2, 0.2), (0.0, 10.0),
                              ng=(10, 8), seed_lo=(-0.9, -0.7), seed_spacing=(0.2, 0.2), t0=0.0, tf=3.0, h=0.1)
    fs = oracle.OracleField.from_workload(ws)
    F, fl, es, cg, ft, te, st = oracle.early_cg(fs, 2, ws.ng, ws.seed_spacing, ws.seed_periodic, ws.period, ws.seeds(), 0.0, 3.0, 0.1, every=5)
    ok = te > 0
    assert (fl == 1).sum() > 10 and len(np.unique(te[ok])) >= 3
    assert np.max(np.abs(ft[ok] - 0.999999233219801983)) <= 1e-9


# -------------------------------------------------------------------------------------------------
# O11 (row f4, first part): Gaussian smoothing of the FTLE field
def test_P18_gaussian_smoothing(oracle):
    """Pins for O11: equal to scipy.ndimage.gaussian_filter1d (mode wrap, truncate 3) applied axis by axis on periodic grids;
    constants are fixed points; the sum is conserved on periodic grids; a linear ramp is reproduced in the interior of a
    non-periodic grid; NaN centres stay NaN and NaN neighbours are skipped with renormalisation; impulse response = weights."""
    from scipy.ndimage import gaussian_filter1d
    rng = np.random.default_rng(18)
    f3 = rng.standard_normal((12, 10, 14))                                 # [z][y][x]
    for sigma in (1.0, 2.0):
        ref = f3
        for ax in (2, 1, 0):                                              # axis 0 of the seed grid is the fastest (last) index
            ref = gaussian_filter1d(ref, sigma, axis=ax, mode="wrap", truncate=3.0)
        out = oracle.smooth_gaussian(3, (14, 10, 12), (1, 1, 1), sigma, f3).reshape(f3.shape)
        assert np.max(np.abs(out - ref)) <= 1e-13
        assert abs(out.sum() - f3.sum()) <= 1e-10
    c = oracle.smooth_gaussian(2, (9, 7), (0, 1), 1.5, np.full(63, 3.25))
    assert np.max(np.abs(c - 3.25)) <= 1e-15
    ramp = np.tile(np.arange(40, dtype=np.float64), (6, 1))               # f = x on a 40 x 6 grid, non-periodic in x
    out = oracle.smooth_gaussian(2, (40, 6), (0, 0), 2.0, ramp).reshape(6, 40)
    assert np.max(np.abs(out[:, 6:-6] - ramp[:, 6:-6])) <= 1e-12 and out[0, 0] > 0.0     # one-sided average at the edge
    imp = np.zeros(21); imp[10] = 1.0
    out = oracle.smooth_gaussian(2, (21, 1), (0, 0), 1.0, imp)
    w = np.exp(-np.arange(-3, 4) ** 2 / 2.0); w /= w.sum()
    assert np.max(np.abs(out[7:14] - w)) <= 1e-15 and np.all(out[:7] == 0) and np.all(out[14:] == 0)
    g = rng.standard_normal(30); g[11] = np.nan
    out = oracle.smooth_gaussian(2, (30, 1), (1, 0), 1.0, g)
    assert np.isnan(out[11]) and np.isfinite(np.delete(out, 11)).all()
    k = np.arange(-3, 4); wk = np.exp(-k ** 2 / 2.0); vals = g[(12 + k) % 30]; ok = np.isfinite(vals)
    assert abs(out[12] - (wk[ok] * vals[ok]).sum() / wk[ok].sum()) <= 1e-15


# -------------------------------------------------------------------------------------------------
# O12 (row f4, second part): Adams-Bashforth 4 with RK4 start-up
def test_P19_adams_bashforth(oracle):
    """Pins for O12.  (a) u = a + b t (time-linear, uniform in space): AB4 integrates cubics in t exactly, RK4 too, and
    linear time interpolation is exact with steps aligned to snapshots: x(T) = x0 + a T + b T^2 / 2.  (b) u = A x: the scheme
    is the linear recurrence x_{n+1} = x_n + (h/24) A (55 x_n - 59 x_{n-1} + 37 x_{n-2} - 9 x_{n-3}) after three P(hA)
    steps; the oracle must reproduce it to rounding.  (c) Fourth order: the error against exp(A T) x0 falls about 16x per
    halving of h.  (d) Exit handling: flags 0/1/2 and frozen positions in an open box."""
    a, b, T = np.array([0.3, -0.2]), np.array([0.05, 0.1]), 4.0
    w = I.analytic_cartesian(2, I.time_linear_uniform(a, b), (9, 9), (-4.0, -4.0), (1.0, 1.0), np.arange(0.0, 5.0, 1.0), ng=(5, 4),
                             seed_lo=(-1.0, -1.0), seed_spacing=(0.3, 0.3), t0=0.0, tf=T, h=0.25)
    fo = oracle.OracleField.from_workload(w)
    F, fl, es = fo.advect_ab4(w.seeds(), 0.0, T, 0.25)
    assert np.all(fl == 0) and np.max(np.abs(F - (w.seeds() + a * T + b * T * T / 2))) <= 1e-13
    A = np.array([[0.1, 0.7], [-0.6, -0.2]])
    def run(h, N):
        wl = I.analytic_cartesian(2, I.linear_flow(A), (81, 81), (-4.0, -4.0), (0.1, 0.1), (0.0, 8.0), ng=(3, 3), seed_lo=(-0.4, -0.3),
                                  seed_spacing=(0.35, 0.3), t0=0.0, tf=h * N, h=h)
        return wl, oracle.OracleField.from_workload(wl).advect_ab4(wl.seeds(), 0.0, h * N, h)
    h, N = 0.05, 40
    wl, (F, fl, es) = run(h, N)
    hA = h * A
    P = np.eye(2) + hA + hA @ hA / 2 + hA @ hA @ hA / 6 + hA @ hA @ hA @ hA / 24
    xs = [wl.seeds().T]
    for n in range(N):
        if n < 3:
            xs.append(P @ xs[-1])
        else:
            xs.append(xs[-1] + (h / 24) * (A @ (55 * xs[-1] - 59 * xs[-2] + 37 * xs[-3] - 9 * xs[-4])))
    assert np.all(fl == 0) and np.max(np.abs(F - xs[-1].T)) <= 1e-13
    from scipy.linalg import expm
    errs = []
    for h, N in ((0.1, 20), (0.05, 40), (0.025, 80)):
        wl, (F, fl, es) = run(h, N)
        errs.append(np.max(np.abs(F - (expm(A * 2.0) @ wl.seeds().T).T)))
    assert 11 <= errs[0] / errs[1] <= 20 and 13 <= errs[1] / errs[2] <= 19
    c = np.array([0.3, 0.13])
    wb = I.analytic_cartesian(2, I.linear_flow(np.zeros((2, 2)), c), (5, 5), (0.0, 0.0), (1.0, 1.0), (0.0, 10.0), ng=(16, 16),
                              seed_lo=(-0.5, -0.5), seed_spacing=(0.31, 0.31), t0=0.0, tf=5.0, h=0.25)
    fb = oracle.OracleField.from_workload(wb)
    F, fl, es = fb.advect_ab4(wb.seeds(), 0.0, 5.0, 0.25)
    assert set(np.unique(fl)) == {0, 1, 2}
    inside = fl != 2
    assert np.max(np.abs(F[inside] - (wb.seeds()[inside] + np.outer(es[inside] * 0.25, c)))) <= 1e-12   # uniform flow: exact until the exit
    assert np.array_equal(F[~inside], wb.seeds()[~inside]) and np.all(es[fl == 2] == 0) and np.all(es[fl == 0] == 20)


# -------------------------------------------------------------------------------------------------
# O13 (row f4, third part): ridges of the smoothed FTLE field
def test_P20_ridge_indicator(oracle):
    """Pins for O13 on analytic fields.  (a) Straight ridge s = exp(-(y - y0)^2 / (2 b^2)): kappa = -s / b^2 on the ridge row,
    n = (0, 1), d = ds/dy, and the mask marks exactly the grid row(s) within half a cell of y0.  (b) Quadratic field
    s = c - (p x^2 + q y^2 + r x y)/2: central differences are exact, so kappa is the smallest eigenvalue of -[[p, r/2],[r/2, q]]
    and d = g . n to rounding.  (c) Circular ridge: the mask is a closed ring of radius R.  (d) Planar ridge sheet in 3D.
    (e) NaN in the stencil or a stencil leaving a non-periodic grid gives NaN / mask 0; a valley (kappa > 0) is not marked."""
    nx, ny, dx, dy = 60, 41, 0.05, 0.04
    X, Y = np.meshgrid((np.arange(nx) + 0.5) * dx, (np.arange(ny) + 0.5) * dy)
    y0, b = 0.83, 0.2
    s = np.exp(-(Y - y0) ** 2 / (2 * b * b))
    kap, d, m = (a.reshape(ny, nx) for a in oracle.ridge(2, (nx, ny), (dx, dy), (0, 0), 0.0, 0.5, s))
    jr = int(np.argmin(np.abs(Y[:, 0] - y0)))
    assert abs(kap[jr, 10] + s[jr, 10] / (b * b)) <= 0.03 / (b * b)                      # O(dy^2) finite-difference error
    rows = np.nonzero(m[:, 10])[0]
    assert set(rows) == set(np.nonzero(np.abs(Y[:, 0] - y0) <= dy / 2 * 1.02)[0]) and len(rows) >= 1
    assert np.all(m[1:-1, 1:-1] == m[1:-1, 10:11])                                       # the same rows at every interior x
    assert np.all(np.isnan(kap[0])) and np.all(np.isnan(kap[:, 0])) and m[0].sum() == 0   # stencil leaves the grid
    p, q, r = 1.3, 0.4, 0.5
    s2 = 2.0 - (p * X * X + q * Y * Y + r * X * Y) / 2
    kap, d, m = (a.reshape(ny, nx) for a in oracle.ridge(2, (nx, ny), (dx, dy), (0, 0), 0.0, -1e9, s2))
    Hm = -np.array([[p, r / 2], [r / 2, q]])
    wv, vv = np.linalg.eigh(Hm)
    nvec = vv[:, 0] * np.sign(vv[np.argmax(np.abs(vv[:, 0])), 0])
    gx, gy = -(p * X + r * Y / 2), -(q * Y + r * X / 2)
    assert np.nanmax(np.abs(kap[1:-1, 1:-1] - wv[0])) <= 1e-10
    assert np.nanmax(np.abs(d[1:-1, 1:-1] - (gx * nvec[0] + gy * nvec[1])[1:-1, 1:-1])) <= 1e-10
    n2 = 81
    Xc, Yc = np.meshgrid((np.arange(n2) - 40) * 0.05, (np.arange(n2) - 40) * 0.05)
    R = np.hypot(Xc, Yc)
    s3 = np.exp(-(R - 1.2) ** 2 / (2 * 0.25 ** 2))
    kap, d, m = (a.reshape(n2, n2) for a in oracle.ridge(2, (n2, n2), (0.05, 0.05), (0, 0), 1.0, 0.8, s3))   # s_min = 0.8 cuts the shoulders beyond the inflection circle, where the
    # tangential curvature s'/r < 0 is the smallest eigenvalue and g . n vanishes identically (a known artefact of height ridges)
    assert m.sum() > 100 and np.all(np.abs(R[m == 1] - 1.2) <= 0.05) and np.all(m[np.abs(R - 1.2) > 0.06] == 0)
    ang = np.arctan2(Yc[m == 1], Xc[m == 1])
    assert np.max(np.diff(np.sort(ang))) < 0.12                                           # a closed ring, no gaps
    nz = 30
    Z = ((np.arange(nz) + 0.5) * 0.1)[:, None, None] * np.ones((nz, 12, 14))
    s4 = np.exp(-(Z - 1.42) ** 2 / (2 * 0.4 ** 2))
    kap, d, m = (a.reshape(nz, 12, 14) for a in oracle.ridge(3, (14, 12, nz), (0.1, 0.1, 0.1), (1, 1, 0), 0.0, 0.5, s4))
    kr = int(np.argmin(np.abs(Z[:, 0, 0] - 1.42)))
    assert np.all(m[kr] == 1) and m.sum() == 12 * 14 and np.all(np.isfinite(kap[1:-1]))   # periodic in x, y: whole sheet
    s5 = s.copy(); s5[20, 30] = np.nan
    kap, d, m = (a.reshape(ny, nx) for a in oracle.ridge(2, (nx, ny), (dx, dy), (0, 0), 0.0, 0.0, s5))
    assert np.all(np.isnan(kap[19:22, 29:32])) and m[19:22, 29:32].sum() == 0 and np.isfinite(kap[20, 33])
    kap, d, m = oracle.ridge(2, (nx, ny), (dx, dy), (0, 0), 0.0, -1e9, -s)
    assert m.reshape(ny, nx)[jr, 5:-5].sum() == 0                                         # a valley is not a ridge
