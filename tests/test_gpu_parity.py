"""GPU parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Gates are BASELINE.json's: bit-exact cell indices; fp64 non-chaotic flow maps
within 1e-10 absolute and FTLE within 1e-8 relative; fp32 / chaotic configs >= 99.9% of seeds within
1e-3 * domain length and median FTLE relative error <= 1e-3.
"""
import numpy as np
import pytest

from paper_2209_13775_b200 import inputs as I
from parity_utils import gate_fp64, gate_statistical, gpu_cg, gpu_run, oracle_cg, oracle_run

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lcs():
    import torch
    assert torch.cuda.is_available()
    from paper_2209_13775_b200 import build, lcs as L
    build.build()
    L.lib()
    return L


def cpu(t):
    return t.detach().cpu().numpy()


# -------------------------------------------------------------------------------------------------
# lcs_locate: bit-exact
def test_locate_cartesian_bit_exact(lcs, oracle):
    import torch
    rng = np.random.default_rng(31)
    for dim, per in ((2, (0, 0)), (3, (0, 0, 0)), (3, (1, 1, 1)), (3, (1, 0, 1))):
        n = (11, 7, 5)[:dim]
        origin, sp = (-1.0, 2.0, 0.5)[:dim], (0.3, 0.25, 0.7)[:dim]
        w = I.analytic_cartesian(dim, lambda p, t: p, n, origin, sp, (0.0, 1.0), ng=(2,) * dim, seed_lo=(0,) * dim,
                                 seed_spacing=(1,) * dim, t0=0.0, tf=1.0, h=0.5, periodic=per)
        lo = np.array(origin)
        hi = lo + (np.array(n) - 1) * np.array(sp)
        pts = rng.uniform(lo - 2.0, hi + 2.0, size=(50000, dim))
        nodes = w.nodes()                                  # points exactly on grid lines / nodes / the closed upper end
        pts = np.concatenate([pts, nodes, nodes + 1e-16, hi[None, :], lo[None, :]])
        fo = oracle.OracleField.from_workload(w)
        co, wo = fo.cart_locate(pts)
        fg = lcs.Field.from_workload(w)
        cg_, wg = fg.locate(torch.from_numpy(pts).cuda(), want_bary=True)
        assert np.array_equal(cpu(cg_), co)
        assert np.array_equal(cpu(wg)[co >= 0], wo[co >= 0])


@pytest.mark.parametrize("dim", [2, 3])
def test_locate_simplex_exact_ties(lcs, oracle, dim):
    """Kuhn mesh with integer coordinates: points exactly on faces, edges and vertices (s == 0 ties)."""
    import torch
    n = 6 if dim == 2 else 5
    V, C = I.kuhn_mesh(dim, n)
    w = I.analytic_simplex(dim, lambda p, t: p, V, C, (0.0, 1.0), ng=(2,) * dim, seed_lo=(0,) * dim,
                           seed_spacing=(1,) * dim, t0=0.0, tf=1.0, h=0.5)
    g = np.arange(0, 2 * (n - 1) + 1) * 0.5
    lattice = np.stack([x.ravel() for x in np.meshgrid(*([g] * dim), indexing="ij")], 1)
    rng = np.random.default_rng(32)
    pts = np.concatenate([lattice, rng.uniform(-0.5, n - 0.5, size=(20000, dim)), lattice[:300] * (2.0 / 3.0)])
    fo = oracle.OracleField.from_workload(w)
    cb, count = fo.locate_brute(pts)
    assert count.max() <= 1
    fg = lcs.Field.from_workload(w)
    cg_, bary = fg.locate(torch.from_numpy(pts).cuda(), want_bary=True)
    assert np.array_equal(cpu(cg_), cb)
    b = cpu(bary)[cb >= 0]
    assert np.allclose(b.sum(1), 1.0, atol=1e-13) and b.min() > -1e-12


@pytest.mark.parametrize("dim", [2, 3])
def test_locate_simplex_delaunay(lcs, oracle, dim):
    """Jittered Delaunay meshes (recipe of configs 2 / 4, reduced): all queries vs the oracle's walk, a
    sample vs brute force; barycentric weights vs the oracle's interpolation of u = x."""
    import torch
    rng = np.random.default_rng(33)
    if dim == 2:
        w = I.config2(ng=(64, 32), lattice=(80, 40))
        lo, hi = np.array([0.0, 0.0]), np.array([2.0, 1.0])
    else:
        w = I.config4(ng=(8, 8, 8), delta=0.08, n_snap=3, length=3.0)
        lo, hi = np.array([-1.0, -1.0, 0.0]), np.array([1.0, 1.0, 3.0])
    fo = oracle.OracleField.from_workload(w)
    pts = np.concatenate([rng.uniform(lo - 0.05, hi + 0.05, size=(200000, dim)),
                          w.vertices[w.cells[:2000, 1:]].mean(axis=1)])       # face centroids: near-ties on one face
    co = fo.locate_walk(pts)
    fg = lcs.Field.from_workload(w)
    cg_, bary = fg.locate(torch.from_numpy(pts).cuda(), want_bary=True)
    cg_ = cpu(cg_)
    assert np.array_equal(cg_, co)
    sub = rng.choice(len(pts), 3000, replace=False)
    cb, count = fo.locate_brute(pts[sub])
    assert count.max() <= 1 and np.array_equal(cb, cg_[sub])
    inside = co >= 0
    assert inside.mean() > 0.5 and (~inside).sum() > 100
    b = cpu(bary)[inside]
    rec = np.einsum("ni,nid->nd", b, w.vertices[w.cells[co[inside]]])
    assert np.max(np.abs(rec - pts[inside])) < 1e-11
    assert fg.info("n_cells") == len(w.cells)
    # adjacency: hull faces counted by the library == faces that appear once
    assert fg.info("n_boundary_faces") == int((fo.neigh < 0).sum())


# -------------------------------------------------------------------------------------------------
# flow map + CG + FTLE parity on the five configs
def test_config1_full_size_fp64(lcs, oracle):
    """Config 1 at BASELINE.json's full size: 201x101 grid, 256x128 seeds, 100 steps, fp64."""
    w = I.config1()
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w)
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    assert np.all(flo == 0) and np.all(eso == 100)                       # closed domain: any exit is a bug
    err = gate_fp64(cpu(F), Fo, cpu(ftg), fto, w.tf - w.t0, cpu(flag), flo, cpu(es), eso)
    assert np.array_equal(cpu(stg), sto)
    assert np.nanmax(np.abs(cpu(cgg) - cgo) / np.maximum(np.abs(cgo), 1.0)) < 1e-7
    print("config1 max flow-map error %.3e mean %.3e" % (err, np.mean(np.linalg.norm(cpu(F) - Fo, axis=1))))


@pytest.mark.parametrize("full", [False, True])
def test_config2_triangles_fp64(lcs, oracle, full):
    """Config 2 (reduced and at BASELINE.json's full size: 50 403 vertices, 1024x512 seeds, 300 steps)."""
    w = I.config2() if full else I.config2(ng=(96, 48), lattice=(60, 30), T=6.0)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w)
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    assert np.all(flo == 0)
    err = gate_fp64(cpu(F), Fo, cpu(ftg), fto, w.tf - w.t0, cpu(flag), flo, cpu(es), eso)
    print("config2 full=%s max flow-map error %.3e" % (full, err))
    if full:
        # SURVEY.md 8.3 parity protocol: lcs_locate bit-exact on ALL seeds against the oracle's walk and on 1e4 sampled seeds
        # against brute force over all cells
        import torch
        pts = w.seeds().astype(np.float64)
        cell = cpu(f.locate(torch.from_numpy(pts).cuda()))
        assert np.array_equal(cell, fo.locate_walk(pts)) and cell.min() >= 0
        sub = np.random.default_rng(22).choice(len(pts), 10000, replace=False)
        cb, count = fo.locate_brute(pts[sub])
        assert count.max() == 1 and np.array_equal(cb, cell[sub]) and f.info("locate_fallbacks") == 0
    assert f.info("walk_cap_hits") == 0


def test_config3_reduced_fp32(lcs, oracle):
    """Config 3 reduced (ABC, periodic 32^3 grid, 48^3 seeds, fp32 data and arithmetic), full oracle comparison."""
    w = I.config3(ngrid=48, nn=32, T=5.0, h=0.01, n_snap=21)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w)
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    assert np.all(cpu(flag) == 0) and np.all(cpu(es) == 500)
    stats = gate_statistical(cpu(F), Fo, cpu(ftg), fto, w.L, cpu(flag), flo)
    print("config3 reduced", stats)


def periodic_block(w, S32, n, B, k0, j0, i0):
    """Seeds of the B^3 block of an n^3 periodic cell-centred seed grid whose lowest index is (i0, j0, k0) (x fastest),
    indices wrapping past n - 1: the stored fp32 seeds, shifted by whole periods so that the block is contiguous in space
    (the field is periodic and positions are never wrapped, reading #13).  Returns (seeds fp64 [B^3][3], wrapped
    flat seed indices [B^3], period shift [B^3][3])."""
    kk, jj, ii = np.meshgrid(k0 + np.arange(B), j0 + np.arange(B), i0 + np.arange(B), indexing="ij")
    idx = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], 1)
    wrapped = idx % n
    flat = wrapped[:, 0] + n * (wrapped[:, 1] + n * wrapped[:, 2])
    shift = (idx // n).astype(np.float64) * np.asarray(w.period, dtype=np.float64)[None, :]
    return S32[flat].astype(np.float64) + shift, flat, shift


def compare_periodic_blocks(oracle, w, fo, F, ftle, blocks, B, t0, tf, h):
    """SURVEY.md 8.3 parity protocol for the periodic 3D configs at full size: the oracle integrates seeded contiguous B^3
    blocks (B - 2 interior + 1-seed halo so that the FTLE is comparable); returns per-seed flow-map errors and per-interior-seed
    relative FTLE errors.  Blocks may straddle the periodic seam of the seed grid (indices wrapping n-1 -> 0): there the GPU's
    FTLE went through lcs_cg_ftle's +-period seam path while the oracle differentiates a contiguous block."""
    n = w.ng[0]
    S32 = w.seeds()
    Fh, fth = cpu(F), cpu(ftle)
    errs, rels = [], []
    for (k0, j0, i0) in blocks:
        blk, flat, shift = periodic_block(w, S32, n, B, k0, j0, i0)
        Fo, flo, _ = fo.advect(blk, t0, tf, h)
        assert np.all(flo == 0)
        errs.append(np.linalg.norm(Fh[flat].astype(np.float64) + shift - Fo, axis=1))
        cgo, fto, sto = oracle.cg_ftle(3, (B, B, B), w.seed_spacing, (0, 0, 0), (0, 0, 0), Fo, flo, tf - t0)
        inner = np.zeros((B, B, B), bool)
        inner[1:-1, 1:-1, 1:-1] = True
        inner = inner.ravel()
        rels.append(np.abs(fth[flat][inner].astype(np.float64) - fto[inner]) / np.maximum(np.abs(fto[inner]), 1e-300))
    return np.concatenate(errs), np.concatenate(rels)


def test_config3_full_size_sampled_blocks(lcs, oracle):
    """Config 3 at full size (128^3 grid, 256^3 seeds, 500 steps) in bench.py's launch configuration (options as bench.py
    leaves them: the defaults).  SURVEY.md 8.3 protocol: the oracle integrates 8 seeded contiguous 34^3 blocks (32^3 + halo);
    two of them straddle the periodic seam of the seed grid on every axis, so the seam path of lcs_cg_ftle is compared at
    full size."""
    w = I.config3()
    f, sd, F, flag, es = gpu_run(w)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    assert int(flag.max()) == 0 and int(es.min()) == 500
    fo = oracle.OracleField.from_workload(w)
    rng = np.random.default_rng(34)
    B = 34
    blocks = [tuple(int(v) for v in rng.integers(0, 256 - B, 3)) for _ in range(6)]
    blocks += [(240, 245, 250), (int(rng.integers(0, 200)), 230, int(rng.integers(0, 200)))]       # wrap 255 -> 0
    err, rel = compare_periodic_blocks(oracle, w, fo, F, ftg, blocks, B, w.t0, w.tf, w.h)
    frac = np.mean(err <= 1e-3 * w.L)
    print("config3 full: %d seeds, frac_ok %.5f median FTLE rel %.3e mean err %.3e max %.3e" % (err.size, frac, np.median(rel), err.mean(), err.max()))
    assert frac >= 0.999 and np.median(rel) <= 1e-3


def test_config4_reduced_tets_fp32(lcs, oracle):
    """Config 4 reduced (pipe, Delaunay tets, fp32 data and arithmetic, bounding-box seeds with flags 0/1/2)."""
    w = I.config4(ng=(24, 24, 40), delta=0.07, T=2.0, h=0.005, n_snap=12, length=4.0)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w)
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    fl = cpu(flag)
    assert (flo == 2).sum() > 100 and (flo == 1).sum() > 100 and (flo == 0).sum() > 100
    assert np.array_equal(fl == 2, flo == 2)                             # initial location is canonical: exact
    stats = gate_statistical(cpu(F), Fo, cpu(ftg), fto, w.L, fl, flo)
    both1 = (fl == 1) & (flo == 1)
    assert np.mean(np.abs(cpu(es)[both1] - eso[both1]) <= 1) > 0.999
    assert f.info("walk_cap_hits") == 0 and f.info("locate_fallbacks") == 0
    print("config4 reduced", stats, "flag mismatches", int((fl != flo).sum()))


@pytest.mark.parametrize("options", [dict(), dict(preblend=1, bundle=1, preblend_steps=9), dict(preblend=1, bundle=1, field_sets=8)])
def test_config5_reduced_backward_streamed(lcs, oracle, options):
    """Config 5 reduced: backward-time windows of the ABC field with a ring of 3 device slots fed from pinned
    host memory on the side stream; results equal the all-resident field bit for bit and pass the gate."""
    import torch
    w = I.config5(ngrid=24, nn=32, n_grids=3, T=2.0, h=0.01, n_snap=9)
    f_ring = lcs.Field.from_workload(w, max_resident_snapshots=3)
    f_all = lcs.Field.from_workload(w)
    for k, v in options.items():
        f_ring.set_option(k, v)
    assert f_ring.info("ring") == 1 and f_all.info("ring") == 0
    fo = oracle.OracleField.from_workload(w)
    s = w.seeds()
    for (t_rel, t_end) in w.meta["windows"]:
        _, _, Fr, flr, esr = gpu_run(w, field=f_ring, t0=t_rel, tf=t_end, h=w.h)
        _, _, Fa, fla, esa = gpu_run(w, field=f_all, t0=t_rel, tf=t_end, h=w.h)
        assert torch.equal(Fr, Fa) and torch.equal(flr, fla)
        Fo, flo, eso = fo.advect(s.astype(np.float64), t_rel, t_end, w.h)
        cgo, fto, sto = oracle_cg(oracle, w, Fo, flo, T=t_end - t_rel)
        cgg, ftg, stg = gpu_cg(w, Fr, flr, T=t_end - t_rel)
        stats = gate_statistical(cpu(Fr), Fo, cpu(ftg), fto, w.L, cpu(flr), flo)
    assert f_ring.info("h2d_bytes") > 0
    if options.get("field_sets"):
        # volumes released one snapshot interval apart share 3 of their 4 windows: resident blended-field sets are reused,
        # and the results above are still bit-identical to the field that blends every chunk
        assert f_ring.info("field_set_hits") >= 6 and f_ring.info("field_set_misses") >= 4
    print("config5 reduced", stats)


@pytest.mark.parametrize("case", ["backward_ring", "forward_chunks", "nonperiodic_exits", "misaligned", "triangles"])
def test_advect_series_identical_to_per_volume_advect(lcs, oracle, case):
    """lcs_advect_series (FTLE time series: the same seeds released at several times): volumes that overlap in time are advanced
    together -- one blend and one integrator launch per snapshot window over the bundled tracers of all of them -- and every
    volume still equals, bit for bit, the lcs_advect of that volume alone (flow map, flags and exit steps: a record carries its
    own step count).  Cases: config 5 reduced (backward, ring of 3 slots, volumes one snapshot interval apart); forward with
    several chunks per window; a non-periodic grid with flags 0/1/2; release times that are not whole snapshot intervals apart
    and a triangle mesh (both integrated volume by volume).  One volume is gated against the oracle."""
    import torch
    opts = dict(bundle=1, preblend=1)
    ring = 0
    if case == "backward_ring":
        w = I.config5(ngrid=24, nn=32, n_grids=6, T=2.0, h=0.01, n_snap=13)
        t_start, T, h, ring = [a for (a, b) in w.meta["windows"]], -2.0, w.h, 3
    elif case == "forward_chunks":
        w = I.config3(ngrid=20, nn=16, T=1.5, h=0.01, n_snap=9)
        t_start, T, h = [0.0, 0.5, 1.0, 2.0], 1.5, 0.01
        opts["preblend_steps"] = 20
    elif case == "nonperiodic_exits":
        A = np.array([[0.03, 0.05, 0.0], [-0.02, 0.04, 0.01], [0.0, -0.03, 0.02]])
        w = I.analytic_cartesian(3, I.linear_flow(A, np.array([0.2, -0.05, 0.1])), (21, 17, 13), (0.0, 0.0, 0.0), (0.1, 0.1, 0.1),
                                 (0.0, 1.0, 2.0, 3.0, 4.0, 5.0), ng=(40, 32, 24), seed_lo=(-0.1, -0.1, -0.1), seed_spacing=(2.2 / 40, 1.8 / 32, 1.4 / 24),
                                 t0=0.0, tf=3.0, h=0.04, vel_dtype=np.float32, compute_dtype=np.float32)
        t_start, T, h = [0.0, 1.0, 2.0], 3.0, 0.04
        opts["preblend_steps"] = 6
    elif case == "misaligned":
        w = I.config3(ngrid=20, nn=16, T=1.0, h=0.01, n_snap=9)
        t_start, T, h = [0.0, 0.3, 0.85], 1.0, 0.01
    else:
        w = I.config2(ng=(48, 24), lattice=(30, 15), T=2.0)
        t_start, T, h, opts = [0.0, 0.5, 1.5], 2.0, w.h, dict()
    f = lcs.Field.from_workload(w, max_resident_snapshots=ring, pinned=bool(ring))
    for k, v in opts.items():
        f.set_option(k, v)
    sd = torch.from_numpy(w.seeds()).cuda()
    Fs, fls, ess = f.advect_series(sd, t_start, T, h)
    torch.cuda.synchronize()
    f1 = lcs.Field.from_workload(w)
    for k, v in opts.items():
        f1.set_option(k, v)
    for k, t0 in enumerate(t_start):
        F, fl, es = f1.advect(sd, t0, t0 + T, h)
        assert torch.equal(Fs[k], F) and torch.equal(fls[k], fl) and torch.equal(ess[k], es), (case, k)
    assert (f.info("series_layers") > 0) == (case in ("backward_ring", "forward_chunks", "nonperiodic_exits"))      # batched or not
    if case == "nonperiodic_exits":
        assert set(np.unique(cpu(fls))) == {0, 1, 2}
    if case == "backward_ring":
        # the host-buffer convenience call returns the same FTLE as cg_ftle on the device results
        fth = f.ftle_series_host(w.ng, w.seed_spacing, w.seed_periodic, w.period, w.seeds(), t_start, T, h)
        for k in range(len(t_start)):
            cgg, ftg, stg = gpu_cg(w, Fs[k].contiguous(), fls[k].contiguous(), T=T)
            assert np.array_equal(fth[k], cpu(ftg), equal_nan=True)
    if case in ("backward_ring", "forward_chunks"):
        k = len(t_start) - 1
        fo = oracle.OracleField.from_workload(w)
        Fo, flo, eso = fo.advect(w.seeds().astype(np.float64), t_start[k], t_start[k] + T, h)
        cgo, fto, sto = oracle_cg(oracle, w, Fo, flo, T=T)
        cgg, ftg, stg = gpu_cg(w, Fs[k].contiguous(), fls[k].contiguous(), T=T)
        gate_statistical(cpu(Fs[k]), Fo, cpu(ftg), fto, w.L, cpu(fls[k]), flo)
    # the series needs a reservation that covers all overlapping volumes
    f2 = lcs.Field.from_workload(w)
    for k, v in opts.items():
        f2.set_option(k, v)
    f2.reserve(sd.shape[0], abs(int(round(T / h))))
    if case in ("backward_ring", "forward_chunks", "nonperiodic_exits"):
        with pytest.raises(lcs.LcsError) as e:
            f2.advect_series(sd, t_start, T, h, reserve=False)
        assert e.value.status == 4


# -------------------------------------------------------------------------------------------------
# closed forms directly on the GPU path, all mesh kinds and dtypes
@pytest.mark.parametrize("mesh", ["cart2", "cart3", "tri", "tet"])
@pytest.mark.parametrize("cdt", [np.float64, np.float32])
def test_linear_flow_closed_form(lcs, oracle, mesh, cdt):
    """u = A x: x_N = P(hA)^N x0 and C = G^T G with G = P(hA)^N (pin P3), for fp64 and fp32 arithmetic."""
    import torch
    from test_oracle_pins import MESHES, P, seedkw
    mk, d = MESHES[mesh]
    rng = np.random.default_rng(21)
    A = rng.normal(size=(d, d)) * 0.25
    A -= np.eye(d) * np.trace(A) / d
    h, N = 0.125, 16
    w = mk(I.linear_flow(A), t0=0.0, tf=h * N, h=h, **seedkw(d))
    if cdt == np.float32:
        w.vel = w.vel.astype(np.float32)
        w.compute_dtype = np.dtype(np.float32)
    f, sd, F, flag, es = gpu_run(w)
    M = np.linalg.matrix_power(P(h * A), N)
    s = w.seeds().astype(np.float64)
    tol = 2e-12 if cdt == np.float64 else 2e-5
    assert np.all(cpu(flag) == 0)
    assert np.max(np.abs(cpu(F) - s @ M.T)) < tol
    cgg, ftg, stg = gpu_cg(w, F, flag)
    Cref = (M.T @ M)[np.triu_indices(d)]
    lam = np.linalg.eigvalsh(M.T @ M)[-1]
    if cdt == np.float64:
        assert np.max(np.abs(cpu(cgg) - Cref)) < 1e-9
        assert np.max(np.abs(cpu(ftg) - np.log(lam) / (2 * h * N))) < 1e-10


def test_mixed_precision_f32_data_f64_arithmetic(lcs, oracle):
    """fp32 velocity storage with fp64 arithmetic: matches the oracle (which widens on read) to the fp64 gate."""
    w = I.config1(ng=(64, 32))
    w.vel = w.vel.astype(np.float32)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w)
    assert np.max(np.abs(cpu(F) - Fo)) < 1e-10
    w3 = I.config3(ngrid=16, nn=16, T=1.0, n_snap=4)
    w3.compute_dtype = np.dtype(np.float64)
    fo, Fo, flo, eso = oracle_run(oracle, w3)
    f, sd, F, flag, es = gpu_run(w3)
    assert np.max(np.abs(cpu(F) - Fo)) < 1e-10


# -------------------------------------------------------------------------------------------------
# edge cases
def test_exit_handling_matches_oracle(lcs, oracle):
    """Open box with uniform flow: flags 0/1/2, exit_step and frozen positions equal the oracle's."""
    for dim in (2, 3):
        c = np.array([0.3, 0.13, -0.07])[:dim]
        w = I.analytic_cartesian(dim, I.linear_flow(np.zeros((dim, dim)), c), (5,) * dim, (0.0,) * dim, (1.0,) * dim,
                                 (0.0, 10.0), ng=(16,) * dim, seed_lo=(-0.5,) * dim, seed_spacing=(0.31,) * dim,
                                 t0=0.0, tf=5.0, h=0.25)
        fo, Fo, flo, eso = oracle_run(oracle, w)
        f, sd, F, flag, es = gpu_run(w)
        assert set(np.unique(flo)) == {0, 1, 2}
        assert np.array_equal(cpu(flag), flo) and np.array_equal(cpu(es), eso)
        assert np.max(np.abs(cpu(F) - Fo)) < 1e-12
        cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
        cgg, ftg, stg = gpu_cg(w, F, flag)
        assert np.array_equal(cpu(stg), sto)
        ok = np.isfinite(fto)
        assert np.array_equal(np.isfinite(cpu(ftg)), ok) and np.allclose(cpu(ftg)[ok], fto[ok], atol=1e-9)


def test_exit_handling_simplex(lcs, oracle):
    w = I.config2(ng=(40, 20), lattice=(30, 15), T=3.0)
    s = I.seed_grid(2, (40, 20, 1), (-0.2, -0.1, 0), (2.4 / 40, 1.2 / 20, 1.0))       # some seeds outside the rectangle
    w.vel = I.sample_field(I.linear_flow(np.zeros((2, 2)), [0.3, 0.05]), w.vertices, w.times, np.float64)
    fo, Fo, flo, eso = oracle_run(oracle, w, seeds=s)
    f, sd, F, flag, es = gpu_run(w, seeds=s)
    assert set(np.unique(flo)) == {0, 1, 2}
    assert np.array_equal(cpu(flag) == 2, flo == 2)
    assert np.mean(cpu(flag) == flo) > 0.995
    same = cpu(flag) == flo
    assert np.max(np.abs(cpu(F)[same] - Fo[same])) < 1e-9
    assert np.mean(np.abs(cpu(es)[same] - eso[same]) <= 1) == 1.0


def test_steps_straddling_snapshots(lcs, oracle):
    """h that does not divide the snapshot spacing: steps straddle snapshot times and each stage time takes
    its own bracket (single-step windows)."""
    w = I.config1(ng=(48, 24), T=6.0, h=0.3)
    fo, Fo, flo, eso = oracle_run(oracle, w, t0=0.35, tf=6.35, h=0.3)
    f, sd, F, flag, es = gpu_run(w, t0=0.35, tf=6.35, h=0.3)
    assert np.max(np.abs(cpu(F) - Fo)) < 1e-10
    assert f.info("windows") > 6
    # backward, fp64
    fo, Fo, flo, eso = oracle_run(oracle, w, t0=6.0, tf=0.0, h=-0.1)
    f, sd, F, flag, es = gpu_run(w, t0=6.0, tf=0.0, h=-0.1)
    assert np.max(np.abs(cpu(F) - Fo)) < 1e-10


def test_argument_errors_and_empty(lcs):
    import torch
    w = I.config1(ng=(8, 4))
    f = lcs.Field.from_workload(w)
    sd = torch.from_numpy(w.seeds()).cuda()
    for (t0, tf, h, status) in ((0.0, 1.0, -0.1, 1), (0.0, 1.0, 0.0, 1), (0.0, 1.0, 0.3, 1), (0.0, 11.0, 0.1, 2), (-1.0, 1.0, 0.1, 2)):
        with pytest.raises(lcs.LcsError) as e:
            f.advect(sd, t0, tf, h)
        assert e.value.status == status, (t0, tf, h, str(e.value))
    F, flag, es = f.advect(sd[:0].contiguous(), 0.0, 1.0, 0.1)
    assert F.shape[0] == 0
    with pytest.raises(lcs.LcsError) as e:
        bad = I.config2(ng=(4, 4), lattice=(6, 5))
        bad.cells = bad.cells.copy()
        bad.cells[3, 1] = 10 ** 6
        lcs.Field.from_workload(bad)
    assert e.value.status == 3
    f2 = lcs.Field(2, 0, w.times, np.float64, np.float64, n=w.n, origin=w.origin, spacing=w.spacing)
    with pytest.raises(lcs.LcsError) as e:
        f2.advect(sd, 0.0, 1.0, 0.1)                                    # snapshots never set
    assert e.value.status == 6


def test_advect_series_arguments_and_single_volume(lcs):
    """lcs_advect_series: argument errors (sign of h against T, interval outside the snapshot times, empty series, resident
    field sets), and a one-volume series, which is lcs_advect."""
    import torch
    w = I.config3(ngrid=16, nn=16, T=1.0, h=0.01, n_snap=5)
    f = lcs.Field.from_workload(w)
    for k, v in dict(bundle=1, preblend=1).items():
        f.set_option(k, v)
    sd = torch.from_numpy(w.seeds()).cuda()
    for (ts, T, h, status) in (([0.0, 0.5], 1.0, -0.01, 1), ([0.0, 0.5], 1.0, 0.0, 1), ([0.0, 1.5], 1.0, 0.01, 2), ([], 1.0, 0.01, 1)):
        with pytest.raises(lcs.LcsError) as e:
            f.advect_series(sd, ts, T, h)
        assert e.value.status == status, (ts, T, h, str(e.value))
    Fs, fls, ess = f.advect_series(sd, [0.5], 1.0, 0.01)
    F, fl, es = f.advect(sd, 0.5, 1.5, 0.01)
    assert f.info("series_layers") == 0 and torch.equal(Fs[0], F) and torch.equal(ess[0], es)
    f.set_option("field_sets", 2)
    with pytest.raises(lcs.LcsError) as e:
        f.advect_series(sd, [0.0, 0.5], 1.0, 0.01)
    assert e.value.status == 1


def test_aliasing_and_host_api(lcs, oracle):
    """flowmap may alias seeds; lcs_ftle_host (host buffers, copies inside the call) equals the device path."""
    import torch
    w = I.config1(ng=(64, 32), T=4.0)
    f, sd, F, flag, es = gpu_run(w)
    sd2 = sd.clone()
    f.advect(sd2, w.t0, w.tf, w.h, flowmap=sd2)
    torch.cuda.synchronize()
    assert torch.equal(sd2, F)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    Fh = np.empty((w.n_seeds, 2))
    flh = np.empty(w.n_seeds, np.uint8)
    ft = f.ftle_host(w.ng, w.seed_spacing, w.seed_periodic, w.period, w.seeds(), w.t0, w.tf, w.h, flowmap=Fh, exit_flag=flh)
    assert np.array_equal(Fh, cpu(F)) and np.array_equal(ft, cpu(ftg), equal_nan=True) and np.array_equal(flh, cpu(flag))


def test_host_api_returns_cg_and_exit_steps(lcs, oracle):
    """lcs_ftle_host with every optional output: Cauchy-Green tensor, exit flags and exit steps equal the device path
    (open box: flags 0 / 1 / 2)."""
    A = np.array([[0.03, 0.05], [-0.02, 0.04]])
    w = I.analytic_cartesian(2, I.linear_flow(A, np.array([0.25, -0.1])), (41, 31), (0.0, 0.0), (0.05, 0.05),
                             (0.0, 2.0, 4.0), ng=(64, 48), seed_lo=(-0.2, -0.1), seed_spacing=(2.4 / 64, 1.7 / 48),
                             t0=0.0, tf=4.0, h=0.05)
    f, sd, F, flag, es = gpu_run(w)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    n = w.n_seeds
    Fh, flh, esh, cgh = np.empty((n, 2)), np.empty(n, np.uint8), np.empty(n, np.int32), np.empty((n, 3))
    ft = f.ftle_host(w.ng, w.seed_spacing, w.seed_periodic, w.period, w.seeds(), w.t0, w.tf, w.h, flowmap=Fh, exit_flag=flh,
                     exit_step=esh, cg=cgh)
    assert set(np.unique(flh)) == {0, 1, 2}
    assert np.array_equal(Fh, cpu(F)) and np.array_equal(flh, cpu(flag)) and np.array_equal(esh, cpu(es))
    assert np.array_equal(ft, cpu(ftg), equal_nan=True) and np.array_equal(cgh, cpu(cgg), equal_nan=True)


def test_reserve_then_hot_calls_do_not_allocate(lcs, oracle):
    """the library allocates its scratch in a set-up call, none inside lcs_advect.  After lcs_field_reserve,
    lcs_advect with growing seed counts (and a different integration length) leaves cudaMemGetInfo unchanged; without a
    covering reservation it returns LCS_ERR_OOM instead of allocating; results do not depend on who reserved."""
    import torch
    w = I.config3(ngrid=64, nn=32, T=1.0, h=0.01, n_snap=5)
    f = lcs.Field.from_workload(w)
    for k, v in (("bundle", 1), ("preblend", 1), ("preblend_steps", 10), ("field_sets", 12)):
        f.set_option(k, v)
    sd = torch.from_numpy(w.seeds()).cuda()
    n = sd.shape[0]
    with pytest.raises(lcs.LcsError) as e:
        f.advect(sd, w.t0, w.tf, w.h, reserve=False)
    assert e.value.status == 4 and "lcs_field_reserve" in str(e.value)
    f.reserve(n, 100)
    outs = [(torch.empty_like(sd[:m]), torch.empty(m, dtype=torch.uint8, device="cuda"), torch.empty(m, dtype=torch.int32, device="cuda"))
            for m in (n // 4, n // 2, n)]
    f.advect(sd[:n // 4], w.t0, w.tf, w.h, flowmap=outs[0][0], exit_flag=outs[0][1], exit_step=outs[0][2], reserve=False)   # loads the kernels
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    scratch0 = f.info("scratch_bytes")
    for (m, tf), (Fm, flm, esm) in zip(((n // 4, 1.0), (n // 2, 0.5), (n, 1.0)), outs):
        f.advect(sd[:m], w.t0, tf, w.h, flowmap=Fm, exit_flag=flm, exit_step=esm, reserve=False)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and f.info("scratch_bytes") == scratch0
    assert f.info("field_set_hits") > 0
    with pytest.raises(lcs.LcsError) as e:
        f.advect(sd, w.t0, 2.0, w.h, reserve=False)                      # 200 steps > the 100 reserved
    assert e.value.status == 4
    f1, sd1, F1, fl1, es1 = gpu_run(w, options=dict(bundle=1, preblend=1, preblend_steps=10))
    assert torch.equal(outs[2][0], F1) and torch.equal(outs[2][2], es1)
    for bad in ((0, 10), (10, 0), (1 << 31, 10), (10, 1 << 24)):
        with pytest.raises(lcs.LcsError) as e:
            f.reserve(*bad)
        assert e.value.status == 1


def test_walk_cap_falls_back_to_the_canonical_locate(lcs, oracle):
    """A step so long that a stage point lies 75 / 150 cells away: the in-advect walk on the per-cell affine maps gives up
    after its hop cap and the tracer is handed to the slow instantiation, which locates the point again with the canonical
    fp64 predicate (counted under walk_fallbacks) and interpolates in its owner -- never in a cell that does not contain
    the point (walk_cap_hits stays 0).  The result matches the oracle, which locates every stage point exactly."""
    w = I.config2(ng=(32, 16), lattice=(300, 150), T=10.0)
    w.vel = I.sample_field(I.linear_flow(np.zeros((2, 2)), [0.1, 0.0]), w.vertices, w.times, np.float64)
    f, sd, F, flag, es = gpu_run(w, t0=0.0, tf=10.0, h=10.0)              # one step: stage points 0.5 and 1.0 domain units away
    assert f.info("walk_fallbacks") > 0 and f.info("walk_cap_hits") == 0 and f.info("locate_fallbacks") == 0
    fo, Fo, flo, eso = oracle_run(oracle, w, t0=0.0, tf=10.0, h=10.0)
    assert set(np.unique(flo)) == {0, 1}
    assert np.array_equal(cpu(flag), flo) and np.array_equal(cpu(es), eso) and np.max(np.abs(cpu(F) - Fo)) < 1e-10
    f2, sd2, F2, flag2, es2 = gpu_run(w, t0=0.0, tf=10.0, h=0.05)
    assert f2.info("walk_cap_hits") == 0 and f2.info("walk_fallbacks") == 0
    fo, Fo, flo, eso = oracle_run(oracle, w, t0=0.0, tf=10.0, h=0.05)
    same = cpu(flag2) == flo
    assert same.mean() > 0.995 and np.max(np.abs(cpu(F2)[same] - Fo[same])) < 1e-9


def test_measured_peaks_are_plausible(lcs):
    """lcs_measure_peak (peaks measured on the box): every kind runs and lands in the range a B200 can
    deliver; bench.py quotes its roofline fractions against these."""
    v = {k: lcs.measure_peak(k) for k in lcs.PEAK_KINDS}
    print("measured peaks:", {k: round(x, 2) for k, x in v.items()})
    assert 40.0 < v["fp32_fma_tflops"] < 90.0 and 15.0 < v["fp64_fma_tflops"] < 45.0
    assert 0.5 < v["launch_us"] < 30.0
    assert 3000.0 < v["hbm_copy_gbs"] < 8500.0
    assert v["l2_seq_gbs"] > v["hbm_copy_gbs"] and v["l2_sector_gbs"] > v["hbm_sector_gbs"] > 300.0
    assert v["l1_gather_line_gbs"] > v["l1_gather_spread_gbs"] and 10000.0 < v["l1_gather_line_gbs"] < 45000.0
    assert 5000.0 < v["smem_records_gbs"] <= 1.05 * v["smem_contiguous_gbs"] < 45000.0
    with pytest.raises(lcs.LcsError) as e:
        lcs.measure_peak(99)
    assert e.value.status == 1


def test_cg_ftle_patterns_vs_oracle(lcs, oracle):
    """lcs_cg_ftle alone on synthetic flow maps: random exit flags (one-sided / NaN patterns), periodic seams,
    2D and 3D, fp64 and fp32 storage, ragged grid sizes."""
    import torch
    rng = np.random.default_rng(35)
    for dim, ng, per in ((2, (37, 19), (0, 0)), (2, (16, 16), (1, 0)), (3, (13, 9, 11), (0, 0, 0)), (3, (8, 8, 8), (1, 1, 1)), (2, (5, 1), (0, 0))):
        n = int(np.prod(ng))
        dx = tuple(rng.uniform(0.1, 0.5, dim))
        period = tuple(ng[a] * dx[a] for a in range(dim))
        s = I.seed_grid(dim, tuple(ng) + (1,) * (3 - dim), (0, 0, 0), dx + (1.0,) * (3 - dim))
        F = s + 0.3 * np.sin(2 * np.pi * s / np.array(period)) @ rng.normal(size=(dim, dim)) + rng.normal(size=s.shape) * 0.01
        flag = (rng.uniform(size=n) < 0.15).astype(np.uint8) * rng.integers(1, 3, n).astype(np.uint8)
        for dt in (np.float64, np.float32):
            Fd = F.astype(dt)
            cgo, fto, sto = oracle.cg_ftle(dim, ng, dx, per, period, Fd.astype(np.float64), flag, 3.0)
            cgg, ftg, stg = lcs.cg_ftle(dim, ng, dx, per, period, torch.from_numpy(Fd).cuda(), torch.from_numpy(flag).cuda(), 3.0)
            assert np.array_equal(cpu(stg), sto)
            ok = np.isfinite(fto)
            assert np.array_equal(np.isfinite(cpu(ftg)), ok)
            tol = 1e-12 if dt == np.float64 else 2e-6
            assert np.allclose(cpu(ftg)[ok], fto[ok], rtol=tol, atol=tol)
            assert np.allclose(cpu(cgg)[ok], cgo[ok], rtol=tol * 10, atol=tol)
        cgn, ftn, _ = lcs.cg_ftle(dim, ng, dx, per, period, torch.from_numpy(F).cuda(), None, 3.0, want_cg=False, want_status=False)
        cgo, fto, sto = oracle.cg_ftle(dim, ng, dx, per, period, F, None, 3.0)
        assert cgn is None and np.allclose(cpu(ftn), fto, rtol=1e-12, atol=1e-12, equal_nan=True)


def test_cg_ftle_float_near_double_root(lcs, oracle):
    """DESIGN.md reading #35: for fp32 outputs the largest eigenvalue comes from an fp32 closed form polished by one fp64 Newton
    step, which is ill-conditioned when the two largest eigenvalues of C nearly coincide; such seeds must take the fp64 closed
    form.  Linear flow maps x -> R diag(s, s (1 + d), s3) x with relative gaps d from 1e-6 to 1e-1 (and an exact double and
    triple root): FTLE within 2e-6 of the oracle on the same float flow map."""
    import torch
    ng = (12, 10, 8)
    dx = (0.05, 0.04, 0.03)
    k, j, i = np.meshgrid(np.arange(ng[2]), np.arange(ng[1]), np.arange(ng[0]), indexing="ij")
    X = np.stack([i * dx[0], j * dx[1], k * dx[2]], axis=-1).reshape(-1, 3)
    rng = np.random.default_rng(35)
    worst = 0.0
    for d in (0.0, 1e-6, 1e-5, 1e-4, 1e-3, 1e-2, 1e-1):
        for s3 in (0.5, 1.0 if d == 0.0 else 0.9):
            Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
            A = Q @ np.diag([1.7, 1.7 * (1.0 + d), 1.7 * s3]) @ np.linalg.qr(rng.standard_normal((3, 3)))[0].T
            F = (X @ A.T).astype(np.float32)
            cgo, fto, sto = oracle.cg_ftle(3, ng, dx, (0, 0, 0), (0.0, 0.0, 0.0), F.astype(np.float64), None, 4.0)
            cgg, ftg, stg = lcs.cg_ftle(3, ng, dx, (0, 0, 0), (0.0, 0.0, 0.0), torch.from_numpy(F).cuda(), None, 4.0)
            ok = np.isfinite(fto)
            assert np.array_equal(np.isfinite(cpu(ftg)), ok)
            err = np.max(np.abs(cpu(ftg)[ok].astype(np.float64) - fto[ok]))
            worst = max(worst, err)
            assert np.allclose(cpu(ftg)[ok], fto[ok], rtol=2e-6, atol=2e-6), (d, s3, err)
    print("cg_ftle float near a double root: worst |dFTLE| = %.2e" % worst)


@pytest.mark.parametrize("case", ["periodic3d_f32", "open3d_f32_flags", "open2d_f64"])
def test_cg_ftle_slabs_with_halo_equal_the_whole_grid(lcs, oracle, case, monkeypatch):
    """One volume across ranks (paper_2209_13775_b200/shard.py): every rank's lcs_cg_ftle on its seed slab extended
    by one halo layer of flow map and flags equals the whole-grid lcs_cg_ftle on the rank's own seeds -- bit for bit on open axes
    (flags 0/1/2 included), to the rounding of F + period in the flow map's type for the layers at a periodic seam.  The ranks are
    emulated one after the other on one GPU: the exchange is replaced by cuts from the global arrays (the exchange itself is
    tested with gloo in tests/test_multi_rank.py)."""
    import torch
    from paper_2209_13775_b200 import shard
    rng = np.random.default_rng(81)
    if case == "periodic3d_f32":
        dim, ng, per, period, dt = 3, (12, 10, 9), (1, 1, 1), (1.2, 1.0, 0.9), np.float32
    elif case == "open3d_f32_flags":
        dim, ng, per, period, dt = 3, (11, 9, 8), (0, 0, 0), (0.0, 0.0, 0.0), np.float32
    else:
        dim, ng, per, period, dt = 2, (16, 13), (0, 0), (0.0, 0.0), np.float64
    dx = tuple(0.1 for _ in range(dim))
    n = int(np.prod(ng))
    idx = np.stack(np.meshgrid(*[np.arange(m) for m in ng[::-1]], indexing="ij"), -1).reshape(-1, dim)[:, ::-1]
    F = (idx * 0.1 + 0.05 * np.sin(3.0 * idx * 0.1 + 0.3) + 0.01 * rng.standard_normal((n, dim))).astype(dt)
    flag = (rng.random(n) < (0.15 if "flags" in case else 0.0)).astype(np.uint8) * rng.integers(1, 3, n).astype(np.uint8)
    Fd, fd = torch.from_numpy(F).cuda(), torch.from_numpy(flag).cuda()
    cg0, ft0, st0 = lcs.cg_ftle(dim, ng, dx, per, period, Fd, fd, 2.0, want_cg=True, want_status=True)
    plane = n // ng[dim - 1]
    F3, f3 = Fd.view(ng[dim - 1], plane, dim), fd.view(ng[dim - 1], plane)
    for world in (1, 2, 3):
        for rank in range(world):
            k0, k1 = shard.slab_range(ng[dim - 1], rank, world)

            def fake_exchange(Fs, fs, r, w, periodic, group=None, k0=k0, k1=k1):
                nz = ng[dim - 1]
                lo = (F3[(k0 - 1) % nz], f3[(k0 - 1) % nz]) if (periodic or k0 > 0) else None
                hi = (F3[k1 % nz], f3[k1 % nz]) if (periodic or k1 < nz) else None
                return lo, hi
            monkeypatch.setattr(shard, "exchange_halo", fake_exchange)
            cg, ft, st = shard.cg_ftle_slab(lcs, dim, ng, dx, per, period, F3[k0:k1].reshape(-1, dim).contiguous(), f3[k0:k1].reshape(-1).contiguous(),
                                            2.0, rank, world, want_cg=True, want_status=True)
            a, b = k0 * plane, k1 * plane
            assert torch.equal(st, st0[a:b]), (case, world, rank)
            if per[dim - 1]:
                ok = torch.isfinite(ft0[a:b])
                assert torch.allclose(ft[ok], ft0[a:b][ok], rtol=2e-5, atol=2e-6) and torch.allclose(cg[ok], cg0[a:b][ok], rtol=2e-4, atol=2e-5)
                inner = slice(plane, (k1 - k0 - 1) * plane)                # layers that do not touch the seam-shifted halo
                if rank not in (0, world - 1) and k1 - k0 > 2:
                    assert torch.equal(ft[inner], ft0[a:b][inner])
            else:
                assert torch.equal(torch.nan_to_num(ft, nan=-1.0), torch.nan_to_num(ft0[a:b], nan=-1.0)), (case, world, rank)
                assert torch.equal(torch.nan_to_num(cg, nan=-1.0), torch.nan_to_num(cg0[a:b], nan=-1.0))


# -------------------------------------------------------------------------------------------------
# integrator variants: re-bundled tracers and the paper's split (one kernel per RK4 stage) design
@pytest.mark.parametrize("options", [dict(bundle=1), dict(bundle=1, bundle_steps=7), dict(bundle=1, ld256=0),
                                     dict(integrator=2, bundle=0), dict(integrator=2, bundle=1, bundle_steps=13)])
def test_cartesian_variants_fp64_identical_to_default(lcs, oracle, options):
    """Config 1 reduced in fp64: every variant (bundling on, odd re-bundling period, 128-bit loads, split stages)
    passes the fp64 gate against the oracle, and results come back in the caller's seed order."""
    w = I.config1(ng=(96, 48), T=10.0)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w, options=options)
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    gate_fp64(cpu(F), Fo, cpu(ftg), fto, w.tf - w.t0, cpu(flag), flo, cpu(es), eso)


@pytest.mark.parametrize("options", [dict(bundle=1, bundle_steps=20), dict(integrator=2, bundle=1), dict(bundle=0, ld256=0),
                                     dict(preblend=1, preblend_steps=7), dict(preblend=1, bundle=1, bundle_steps=20)])
def test_config3_variants_fp32(lcs, oracle, options):
    """Config 3 reduced (periodic, fp32) with bundling / split stages: statistical gate; fused variants that differ
    only in tracer order are bit-identical to the default path (a tracer's arithmetic does not depend on its slot)."""
    w = I.config3(ngrid=40, nn=32, T=2.0, h=0.01, n_snap=9)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f0, sd0, F0, flag0, es0 = gpu_run(w, options=dict(bundle=0))
    f, sd, F, flag, es = gpu_run(w, options=options)
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    gate_statistical(cpu(F), Fo, cpu(ftg), fto, w.L, cpu(flag), flo)
    if options.get("integrator", 0) != 2:
        assert np.array_equal(cpu(F), cpu(F0))


@pytest.mark.parametrize("options", [dict(tma=1), dict(tma=1, tma_cap=96), dict(tma=1, preblend_steps=5, bundle_steps=5), dict(tma=2, bundle_order=1)])
def test_config3_staged_tma_variant_identical(lcs, oracle, options):
    """Row (g): the pre-blended integrator with the stage-time fields staged through shared memory by TMA bulk copies
    (option tma; BASELINE.json north_star, second subsystem).  Same arithmetic on the same records, so the flow map is
    bit-identical to the global-memory gather in every mix of staged steps, steps whose box exceeds the tile capacity
    (tma_cap=96) and re-bundling cadence; statistical gate against the oracle.  On a grid that is not periodic with
    power-of-two node counts the option is ignored (the global-memory kernel runs)."""
    w = I.config3(ngrid=48, nn=32, T=2.0, h=0.01, n_snap=9)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f0, sd0, F0, flag0, es0 = gpu_run(w, options=dict(bundle=1, preblend=1))
    f, sd, F, flag, es = gpu_run(w, options=dict(bundle=1, preblend=1, **options))
    assert np.array_equal(cpu(F), cpu(F0)) and np.array_equal(cpu(es), cpu(es0)) and int(cpu(flag).max()) == 0
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    gate_statistical(cpu(F), Fo, cpu(ftg), fto, w.L, cpu(flag), flo)
    w2 = I.config3(ngrid=24, nn=24, T=0.5, h=0.01, n_snap=3)            # 24 nodes per axis: not a power of two
    fa, sa, Fa, fla, esa = gpu_run(w2, options=dict(bundle=1, preblend=1))
    fb, sb, Fb, flb, esb = gpu_run(w2, options=dict(bundle=1, preblend=1, **options))
    assert np.array_equal(cpu(Fa), cpu(Fb))


@pytest.mark.parametrize("options", [dict(bundle=1, bundle_steps=5), dict(integrator=2, bundle=1)])
def test_exit_handling_variants(lcs, oracle, options):
    """Exits (flags 0/1/2, exit_step) with re-bundling (finished tracers are parked in the last bin) and with the
    split stages (flag raised by the failing stage, record frozen at the start of the step)."""
    A = np.array([[0.03, 0.05], [-0.02, 0.04]])
    w = I.analytic_cartesian(2, I.linear_flow(A, np.array([0.25, -0.1])), (41, 31), (0.0, 0.0), (0.05, 0.05),
                             (0.0, 2.0, 4.0), ng=(64, 48), seed_lo=(-0.2, -0.1), seed_spacing=(2.4 / 64, 1.7 / 48),
                             t0=0.0, tf=4.0, h=0.05)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f, sd, F, flag, es = gpu_run(w, options=options)
    assert (flo == 0).sum() > 20 and (flo == 1).sum() > 100 and (flo == 2).sum() > 20
    assert np.array_equal(cpu(flag), flo) and np.array_equal(cpu(es), eso)
    assert np.max(np.abs(cpu(F) - Fo)) <= 1e-10


def test_preblend_nonperiodic_3d_fp32_with_exits(lcs, oracle):
    """Pre-blended x-pair gathers on a non-periodic 3D fp32 grid with exits (flags 0/1/2) and a step size that makes
    some steps straddle snapshots (those windows fall back to pair records): bit-identical to the pair-record path."""
    A = np.array([[0.05, 0.3, 0.0], [-0.3, 0.02, 0.1], [0.0, -0.1, 0.04]])
    w = I.analytic_cartesian(3, I.linear_flow(A, np.array([0.2, -0.05, 0.1])), (21, 17, 13), (0.0, 0.0, 0.0), (0.1, 0.1, 0.1),
                             (0.0, 1.0, 2.0, 3.0), ng=(40, 32, 24), seed_lo=(-0.1, -0.1, -0.1), seed_spacing=(2.2 / 40, 1.8 / 32, 1.4 / 24),
                             t0=0.0, tf=3.0, h=0.04, vel_dtype=np.float32, compute_dtype=np.float32)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f0, sd0, F0, flag0, es0 = gpu_run(w, options=dict(preblend=0, bundle=0))
    f1, sd1, F1, flag1, es1 = gpu_run(w, options=dict(preblend=1, bundle=1, preblend_steps=6))
    assert set(np.unique(flo)) == {0, 1, 2}
    assert np.array_equal(cpu(F0), cpu(F1)) and np.array_equal(cpu(flag0), cpu(flag1)) and np.array_equal(cpu(es0), cpu(es1))
    assert np.mean(cpu(flag1) == flo) > 0.995
    same = cpu(flag1) == flo
    assert np.max(np.linalg.norm(cpu(F1)[same].astype(np.float64) - Fo[same], axis=1)) < 1e-3 * w.L


@pytest.mark.parametrize("mesh", ["tri_f64", "tet_f32"])
def test_simplex_split_stages_vs_oracle_and_fused(lcs, oracle, mesh):
    """The paper's split design on unstructured meshes (one short kernel per cell search and per interpolation,
    8 launches per RK4 step; integrator option 2): same per-evaluation arithmetic as the fused kernel, so the flow map equals
    the fused one bit for bit wherever the walks end in the same cells (everywhere but within the walk tolerance of a face),
    and passes the gate of its config against the oracle."""
    if mesh == "tri_f64":
        w = I.config2(ng=(96, 48), lattice=(40, 20), T=4.0)
    else:
        w = I.config4(ng=(20, 20, 36), delta=0.08, T=1.5, h=0.005, n_snap=10, length=4.0)
    fo, Fo, flo, eso = oracle_run(oracle, w)
    f1, sd1, F1, flag1, es1 = gpu_run(w, options=dict(integrator=1, bundle=0))
    for opts in (dict(integrator=2, bundle=0), dict(integrator=2, bundle=1, bundle_steps=9)):
        f2, sd2, F2, flag2, es2 = gpu_run(w, options=opts)
        assert f2.info("walk_cap_hits") == 0 and f2.info("locate_fallbacks") == 0
        assert np.mean(cpu(flag2) == cpu(flag1)) > 0.999
        same = (cpu(flag2) == flo)
        if mesh == "tri_f64":
            assert same.mean() > 0.995 and np.max(np.abs(cpu(F2)[same] - Fo[same])) < 1e-9
            assert np.max(np.abs(cpu(F2) - cpu(F1))[cpu(flag2) == cpu(flag1)]) < 1e-9
        else:
            err = np.linalg.norm(cpu(F2).astype(np.float64) - Fo, axis=1)
            assert np.mean((err <= 1e-3 * w.L) & same) >= 0.999


@pytest.mark.parametrize("options", [dict(bundle=1), dict(bundle=1, bundle_steps=7)])
def test_simplex_bundled_identical_to_unbundled(lcs, oracle, options):
    """Re-bundling tracers by bin (triangles fp64, tets fp32 with flags 0/1/2): a tracer's arithmetic does not depend on
    its slot, so results are bit-identical to the unbundled run and come back in the caller's order."""
    import torch
    for w in (I.config2(ng=(96, 48), lattice=(40, 20), T=4.0), I.config4(ng=(20, 20, 36), delta=0.08, T=1.5, h=0.005, n_snap=10, length=4.0)):
        f0, sd0, F0, flag0, es0 = gpu_run(w, options=dict(bundle=0))
        f1, sd1, F1, flag1, es1 = gpu_run(w, options=options)
        assert torch.equal(F0, F1) and torch.equal(flag0, flag1) and torch.equal(es0, es1)
        assert f1.info("locate_fallbacks") == 0 and f1.info("walk_cap_hits") == 0 and f0.info("walk_cap_hits") == 0


@pytest.mark.slow
def test_config4_full_size_sampled(lcs, oracle):
    """Config 4 at full size (2.01 M vertices / 13.4 M tets, 256x256x512 box seeds, 1600 steps) in bench.py's launch
    configuration (bundling on by default at this size).  lcs_locate: bit-exact against the oracle's walk on 2e5 sampled
    seeds and against brute force over all cells on 256 of them, with no fallback.  Flow map / FTLE: the oracle integrates
    10 seeded random 16^3 blocks of the box grid; statistical gate of BASELINE.json with flag mismatches counted as
    failures; the in-advect walk never hits its hop cap."""
    import torch
    w = I.config4()
    f = lcs.Field.from_workload(w)
    fo = oracle.OracleField.from_workload(w)
    seeds = w.seeds()
    rng = np.random.default_rng(44)
    pick = rng.choice(seeds.shape[0], 200000, replace=False)
    pts = np.ascontiguousarray(seeds[pick].astype(np.float64))
    cg_ = cpu(f.locate(torch.from_numpy(pts).cuda()))
    assert np.array_equal(cg_, fo.locate_walk(pts))
    cb, count = fo.locate_brute(pts[:256])
    assert np.array_equal(cg_[:256], cb) and np.all(count <= 1)
    assert f.info("locate_fallbacks") == 0
    sd = torch.from_numpy(seeds).cuda()
    F, flag, es = f.advect(sd, w.t0, w.tf, w.h)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    torch.cuda.synchronize()
    fb = f.info("walk_fallbacks")
    print("config4 full: in-advect walks re-located with the canonical predicate: %d" % fb)
    assert f.info("locate_fallbacks") == 0 and f.info("walk_cap_hits") == 0 and fb < 1e-3 * seeds.shape[0]
    nx, ny, nz = w.ng
    Fh = cpu(F).reshape(nz, ny, nx, 3); fth = cpu(ftg).reshape(nz, ny, nx); flh = cpu(flag).reshape(nz, ny, nx)
    S = seeds.reshape(nz, ny, nx, 3)
    B = 16
    errs, rels, mism, flag_mism, tot, counts = [], [], 0, 0, 0, np.zeros(3, int)
    for b in range(10):
        k0, j0, i0 = int(rng.integers(0, nz - B)), int(rng.integers(0, ny - B)), int(rng.integers(0, nx - B))
        blk = np.ascontiguousarray(S[k0:k0 + B, j0:j0 + B, i0:i0 + B].reshape(-1, 3))
        Fo, flo, eso = fo.advect(blk.astype(np.float64), w.t0, w.tf, w.h)
        Fg = Fh[k0:k0 + B, j0:j0 + B, i0:i0 + B].reshape(-1, 3).astype(np.float64)
        fg = flh[k0:k0 + B, j0:j0 + B, i0:i0 + B].ravel()
        assert np.array_equal(fg == 2, flo == 2)                         # the seeds' cells are canonical: exact
        bad = (np.linalg.norm(Fg - Fo, axis=1) > 1e-3 * w.L) | (fg != flo)
        mism += int(bad.sum()); flag_mism += int((fg != flo).sum()); tot += bad.size
        counts += np.bincount(flo, minlength=3)[:3]
        errs.append(np.linalg.norm(Fg - Fo, axis=1)[fg == flo])
        cgo, fto, sto = oracle.cg_ftle(3, (B, B, B), w.seed_spacing, (0, 0, 0), (0, 0, 0), Fo, flo, w.tf - w.t0)
        fto = fto.reshape(B, B, B)[1:-1, 1:-1, 1:-1]
        ftb = fth[k0 + 1:k0 + B - 1, j0 + 1:j0 + B - 1, i0 + 1:i0 + B - 1].astype(np.float64)
        ok = np.isfinite(fto) & np.isfinite(ftb)
        rels.append((np.abs(ftb[ok] - fto[ok]) / np.maximum(np.abs(fto[ok]), 1e-300)).ravel())
    err = np.concatenate(errs); rel = np.concatenate(rels)
    print("config4 full: %d seeds (flags 0/1/2: %s), frac_ok %.5f, flag mismatches %d, median FTLE rel %.3e (n=%d) mean err %.3e max %.3e" %
          (tot, counts.tolist(), 1 - mism / tot, flag_mism, np.median(rel) if rel.size else 0.0, rel.size, err.mean(), err.max()))
    assert counts.min() > 500                                            # the sample holds stayers, leavers and outside seeds
    assert 1 - mism / tot >= 0.999
    assert rel.size > 500 and np.median(rel) <= 1e-3


@pytest.mark.slow
def test_config5_full_size_series_with_field_sets(lcs, oracle):
    """Config 5 at full size in the configuration bench.py times: ring of 4 device slots fed from pinned host memory and 12
    resident sets of blended fields.  Three consecutive volumes (192^3 seeds, backward 500 steps) on ONE field: the later
    volumes reuse the sets cached by the earlier ones (9 of their 10 windows).  The last volume must equal, bit for bit, the
    same volume from a fresh field WITHOUT field sets, and passes the statistical gate against 6 seeded 18^3 oracle blocks,
    one of them across the periodic seam."""
    import torch
    w = I.config5()
    f = lcs.Field.from_workload(w, max_resident_snapshots=4, pinned=True)
    f.set_option("field_sets", 12)
    sd = torch.from_numpy(w.seeds()).cuda()
    vols = w.meta["windows"][6:9]
    for (t_rel, t_end) in vols:
        F, flag, es = f.advect(sd, t_rel, t_end, w.h)
    cgg, ftg, stg = gpu_cg(w, F, flag, T=t_end - t_rel)
    torch.cuda.synchronize()
    hits, misses = f.info("field_set_hits"), f.info("field_set_misses")
    print("config5 field sets: hits %d misses %d" % (hits, misses))
    assert hits == 18 and misses == 12                                   # 10 windows per volume, 9 shared with the previous one
    assert int(flag.max()) == 0 and f.info("ring") == 1 and f.info("h2d_bytes") > 0
    f.close()
    f0 = lcs.Field.from_workload(w, max_resident_snapshots=4, pinned=True)
    F0, flag0, es0 = f0.advect(sd, t_rel, t_end, w.h)
    torch.cuda.synchronize()
    assert f0.info("field_set_hits") == 0 and torch.equal(F0, F) and torch.equal(flag0, flag) and torch.equal(es0, es)
    f0.close()
    fo = oracle.OracleField.from_workload(w)
    rng = np.random.default_rng(55)
    B = 18
    n = w.ng[0]
    blocks = [tuple(int(v) for v in rng.integers(0, n - B, 3)) for _ in range(5)] + [(n - 9, n - 5, n - 12)]
    err, rel = compare_periodic_blocks(oracle, w, fo, F, ftg, blocks, B, t_rel, t_end, w.h)
    frac = np.mean(err <= 1e-3 * w.L)
    print("config5 full (volume 8 of a 3-volume series): frac_ok %.5f median FTLE rel %.3e mean err %.3e max %.3e" % (frac, np.median(rel), err.mean(), err.max()))
    assert frac >= 0.999 and np.median(rel) <= 1e-3


@pytest.mark.slow
def test_config5_full_size_advect_series(lcs, oracle):
    """Config 5 at full size as bench.py times it by default: lcs_advect_series on a ring of 4 device slots fed from pinned host
    memory.  Four consecutive volumes (192^3 seeds each, backward 500 steps, released one snapshot interval apart) advanced
    together: up to four volumes share a launch.  The first and the last volume must equal, bit for bit, the lcs_advect of that
    volume alone on a fresh field; the last one passes the statistical gate against 6 seeded 18^3 oracle blocks, one of them
    across the periodic seam."""
    import torch
    w = I.config5()
    f = lcs.Field.from_workload(w, max_resident_snapshots=4, pinned=True)
    sd = torch.from_numpy(w.seeds()).cuda()
    vols = w.meta["windows"][5:9]
    t_start = [a for (a, b) in vols]
    T = vols[0][1] - vols[0][0]
    Fs, fls, ess = f.advect_series(sd, t_start, T, w.h)
    torch.cuda.synchronize()
    assert f.info("series_layers") == 13 and f.info("ring") == 1 and f.info("h2d_bytes") > 0 and int(fls.max()) == 0
    f0 = lcs.Field.from_workload(w, max_resident_snapshots=4, pinned=True)
    for k in (0, 3):
        F0, flag0, es0 = f0.advect(sd, t_start[k], t_start[k] + T, w.h)
        assert torch.equal(F0, Fs[k]) and torch.equal(flag0, fls[k]) and torch.equal(es0, ess[k]), k
    f0.close()
    F, flag = Fs[3].contiguous(), fls[3].contiguous()
    cgg, ftg, stg = gpu_cg(w, F, flag, T=T)
    fo = oracle.OracleField.from_workload(w)
    rng = np.random.default_rng(56)
    B = 18
    n = w.ng[0]
    blocks = [tuple(int(v) for v in rng.integers(0, n - B, 3)) for _ in range(5)] + [(n - 9, n - 5, n - 12)]
    err, rel = compare_periodic_blocks(oracle, w, fo, F, ftg, blocks, B, t_start[3], t_start[3] + T, w.h)
    frac = np.mean(err <= 1e-3 * w.L)
    print("config5 full (lcs_advect_series, volume 8 of 4): frac_ok %.5f median FTLE rel %.3e mean err %.3e max %.3e" % (frac, np.median(rel), err.mean(), err.max()))
    assert frac >= 0.999 and np.median(rel) <= 1e-3
    f.close()


# -------------------------------------------------------------------------------------------------
# row f2: full eigen-decomposition of C
@pytest.mark.parametrize("dim", [2, 3])
@pytest.mark.parametrize("dt", [np.float64, np.float32])
def test_cg_eigen_vs_oracle(lcs, oracle, dim, dt):
    """lcs_cg_eigen against oracle rule O8 on (i) C of a real flow map (config 1 / config 3 reduced, NaN rows included) and
    (ii) random SPD matrices with condition numbers up to 1e10 (fp64) / 1e4 (fp32).  Eigenvalues within 1e-12 (fp64) or 2e-6
    (fp32) of lambda_max; eigenvectors: residual |C v - lambda v| small, and equal to the oracle's up to rounding where the
    eigenvalue is separated from the others (elsewhere any orthonormal basis of the eigenspace is correct)."""
    import torch
    rng = np.random.default_rng(160 + dim)
    w = I.config1(ng=(64, 32), T=5.0) if dim == 2 else I.config3(ngrid=20, nn=16, T=1.0, n_snap=4)
    f, sd, F, flag, es = gpu_run(w)
    flag = flag.clone(); flag[::97] = 1                                     # some undefined seeds -> NaN rows
    cgg, _, _ = gpu_cg(w, F, flag)
    lc = 10 if dt == np.float64 else 4
    from test_oracle_pins import _random_spd, _sym_from_upper
    mats = np.concatenate([cpu(cgg).astype(np.float64), _random_spd(rng, dim, 4000, lc)]).astype(dt)
    ev_g, vec_g = lcs.cg_eigen(dim, torch.from_numpy(mats).cuda())
    torch.cuda.synchronize()
    ev_g, vec_g = cpu(ev_g).astype(np.float64), cpu(vec_g).astype(np.float64)
    ev_o, vec_o = oracle.cg_eigen(dim, mats.astype(np.float64))
    nanrow = np.isnan(ev_o[:, 0])
    assert nanrow.sum() > 5 and np.array_equal(np.isnan(ev_g[:, 0]), nanrow) and np.all(np.isnan(vec_g[nanrow]))
    ok = ~nanrow
    scale = np.abs(ev_o[ok]).max(axis=1, keepdims=True)
    tol = 1e-12 if dt == np.float64 else 2e-6
    assert np.max(np.abs(ev_g[ok] - ev_o[ok]) / scale) <= tol
    checked = 0
    for i in np.nonzero(ok)[0][::7]:
        a = _sym_from_upper(dim, mats[i].astype(np.float64))
        s = np.abs(ev_o[i]).max()
        for k in range(dim):
            assert np.linalg.norm(a @ vec_g[i, k] - ev_g[i, k] * vec_g[i, k]) <= 10 * tol * s
            gap = min(abs(ev_o[i, k] - ev_o[i, m]) for m in range(dim) if m != k)
            if gap > 1e-2 * s:
                assert np.max(np.abs(vec_g[i, k] - vec_o[i, k])) <= (1e-9 if dt == np.float64 else 2e-4)
                checked += 1
    assert checked > 500


def test_cg_eigen_arguments(lcs):
    import torch
    z = torch.zeros((0, 6), device="cuda")
    ev, vec = lcs.cg_eigen(3, z)
    assert ev.shape == (0, 3) and vec.shape == (0, 3, 3)
    with pytest.raises(lcs.LcsError):
        lcs._check(lcs.lib().lcs_cg_eigen(4, 0, 1, 1, 1, 1, None))


# -------------------------------------------------------------------------------------------------
# row f3: Cauchy-Green tensor from auxiliary points
@pytest.mark.parametrize("case", ["cart2_f64", "tet_f32"])
def test_cg_ftle_aux_vs_oracle(lcs, oracle, case):
    """lcs_cg_ftle_aux against oracle rule O9: the auxiliary tracers are advected by lcs_advect (GPU) and by the oracle, then
    differenced by each side.  fp64 double gyre: fp64 gate; fp32 pipe on tets with exits: statistical FTLE gate and equal
    status wherever both sides agree on the flags of the auxiliary tracers."""
    import torch
    if case == "cart2_f64":
        w = I.config1(ng=(48, 24), T=5.0)
        delta = (1e-3, 1e-3)
    else:
        w = I.config4(ng=(16, 16, 24), delta=0.08, T=1.0, h=0.005, n_snap=8, length=4.0)
        delta = (2e-2, 2e-2, 2e-2)
    dim, T = w.dim, w.tf - w.t0
    aux = I.aux_seeds(w.seeds(), delta).reshape(-1, dim)
    fo, Fo, flo, eso = oracle_run(oracle, w, seeds=aux)
    f, sd, F, flag, es = gpu_run(w, seeds=aux)
    cgo, fto, sto = oracle.cg_ftle_aux(dim, delta, Fo, flo, T)
    cgg, ftg, stg = lcs.cg_ftle_aux(dim, delta, F.reshape(-1, 2 * dim, dim), flag.reshape(-1, 2 * dim), T)
    torch.cuda.synchronize()
    cgg, ftg, stg = cpu(cgg).astype(np.float64), cpu(ftg).astype(np.float64), cpu(stg)
    if case == "cart2_f64":
        assert np.array_equal(cpu(flag), flo) and np.array_equal(stg, sto) and np.all(sto == 0)
        assert np.max(np.abs(cpu(F) - Fo)) <= 1e-10
        assert np.all(np.abs(ftg - fto) <= 1e-8 * np.abs(fto) + 1e-6)       # (1e-10 / delta) / (2 T): the quotient amplifies 1e-10
        assert np.max(np.abs(cgg - cgo) / np.maximum(np.abs(cgo), 1.0)) <= 1e-5
    else:
        same = np.all(cpu(flag).reshape(-1, 2 * dim) == flo.reshape(-1, 2 * dim), axis=1)
        assert same.mean() > 0.99 and np.array_equal(stg[same], sto[same])
        assert (sto == 1).sum() > 50 and (sto == 0).sum() > 200
        ok = same & (sto == 0)
        assert np.all(np.isnan(ftg[same & (sto == 1)]))
        # fp32 positions (1e-7 relative of L = 4) differenced over 2 delta = 0.04: FTLE absolute error budget 1e-4 / T
        assert np.median(np.abs(ftg[ok] - fto[ok])) <= 2e-3
    # the exact same device buffers through the oracle's arithmetic: the kernel's own differencing / eigenvalue is tight
    cgx, ftx, stx = oracle.cg_ftle_aux(dim, delta, cpu(F).astype(np.float64), cpu(flag), T)
    okx = stx == 0
    assert np.array_equal(stg, stx)
    assert np.max(np.abs(ftg[okx] - ftx[okx])) <= (1e-12 if case == "cart2_f64" else 2e-5)


def test_cg_ftle_aux_arguments(lcs):
    import torch
    z = torch.zeros((4, 4, 2), device="cuda", dtype=torch.float64)
    with pytest.raises(lcs.LcsError):
        lcs.cg_ftle_aux(2, (0.0, 1e-3), z, None, 1.0)
    with pytest.raises(lcs.LcsError):
        lcs.cg_ftle_aux(2, (1e-3, 1e-3), z, None, 0.0)
    cg, ft, st = lcs.cg_ftle_aux(2, (1e-3, 1e-3), torch.zeros((0, 4, 2), device="cuda", dtype=torch.float64), None, 1.0)
    assert ft.shape == (0,)


# -------------------------------------------------------------------------------------------------
# row f1: early evaluation of C when a stencil member leaves
@pytest.mark.parametrize("case", ["cart2_f64_open_box", "cart3_f32_preblend", "tet_f32_pipe"])
def test_advect_early_cg_vs_oracle(lcs, oracle, case):
    """lcs_advect_early_cg against oracle rule O10: same evaluation points, same update rule.  fp64 open box (a rotating strain
    flow that pushes tracers out): flags, exit steps and t_eff identical, FTLE within the fp64 gate.  fp32 cases (non-periodic 3D
    grid through the bundled pre-blended integrator; pipe flow on tets): t_eff identical wherever the flags of the whole stencil
    agree, median FTLE error within the statistical gate."""
    import torch
    if case == "cart2_f64_open_box":
        A = np.array([[0.25, 0.6], [-0.6, 0.25]])
        w = I.analytic_cartesian(2, I.linear_flow(A), (41, 41), (-2.0, -2.0), (0.1, 0.1), (0.0, 2.0, 4.0), ng=(24, 20), seed_lo=(-2.1, -1.4),
                                 seed_spacing=(0.175, 0.14), t0=0.0, tf=4.0, h=0.05)      # first and last seed columns lie outside
        every, opts = 7, dict(bundle=1, bundle_steps=11)
    elif case == "cart3_f32_preblend":
        A = np.array([[0.05, 0.3, 0.0], [-0.3, 0.02, 0.1], [0.0, -0.1, 0.04]])
        w = I.analytic_cartesian(3, I.linear_flow(A, np.array([0.2, -0.05, 0.1])), (21, 17, 13), (0.0, 0.0, 0.0), (0.1, 0.1, 0.1),
                                 (0.0, 1.0, 2.0, 3.0), ng=(24, 20, 16), seed_lo=(0.1, 0.1, 0.1), seed_spacing=(1.8 / 24, 1.4 / 20, 1.0 / 16),
                                 t0=0.0, tf=3.0, h=0.05, vel_dtype=np.float32, compute_dtype=np.float32)
        every, opts = 10, dict(bundle=1, preblend=1, preblend_steps=6)
    else:
        w = I.config4(ng=(20, 20, 32), delta=0.08, T=1.5, h=0.005, n_snap=10, length=4.0)
        every, opts = 40, dict(bundle=1, bundle_steps=60)
    fo = oracle.OracleField.from_workload(w)
    args = (w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period)
    Fo, flo, eso, cgo, fto, teo, sto = oracle.early_cg(fo, *args, w.seeds().astype(np.float64), w.t0, w.tf, w.h, every)
    f = lcs.Field.from_workload(w)
    for k, v in opts.items():
        f.set_option(k, v)
    sd = torch.from_numpy(w.seeds()).cuda()
    F, flag, es, cg, ft, te, stt = lcs.advect_early_cg(f, w.ng, w.seed_spacing, w.seed_periodic, w.period, sd, w.t0, w.tf, w.h, every)
    torch.cuda.synchronize()
    F2, flag2, es2 = f.advect(sd, w.t0, w.tf, w.h)                       # the plain call gives the same flow map
    assert torch.equal(F, F2) and torch.equal(flag, flag2) and torch.equal(es, es2)
    flag, es, ft, te, stt = cpu(flag), cpu(es), cpu(ft).astype(np.float64), cpu(te).astype(np.float64), cpu(stt)
    early = (teo > 0) & (teo < (w.tf - w.t0) - 1e-9)
    assert (flo == 1).sum() > 50 and early.sum() > 30 and (teo == 0).sum() > 0
    if case == "cart2_f64_open_box":
        assert np.array_equal(flag, flo) and np.array_equal(es, eso)
        assert np.allclose(te, teo, atol=1e-12) and np.array_equal(stt, sto)
        ok = teo > 0
        assert np.all(np.abs(ft[ok] - fto[ok]) <= 1e-8 * np.abs(fto[ok]) + 1e-10 / teo[ok])
        assert np.all(np.isnan(ft[~ok]))
        assert np.max(np.abs(cpu(cg)[ok] - cgo[ok]) / np.maximum(np.abs(cgo[ok]), 1.0)) <= 1e-9
    else:
        g = [int(w.ng[a]) for a in range(3)]
        agree = (flag == flo) & ((flag != 1) | (es == eso))
        a3 = agree.reshape(g[2], g[1], g[0])
        sten = a3.copy()
        for ax in range(3):
            for sh in (1, -1):
                r = np.roll(a3, sh, axis=ax)
                sl = [slice(None)] * 3; sl[ax] = 0 if sh == 1 else -1
                r[tuple(sl)] = True
                sten &= r
        sten = sten.ravel()
        assert sten.mean() > 0.97
        assert np.allclose(te[sten], teo[sten], atol=1e-5)
        ok = sten & (teo > 0) & np.isfinite(fto)
        assert np.array_equal(np.isfinite(ft[sten]), np.isfinite(fto[sten]))
        rel = np.abs(ft[ok] - fto[ok]) / np.maximum(np.abs(fto[ok]), 1e-3)
        assert np.median(rel) <= 1e-3


def test_advect_early_cg_arguments(lcs):
    import torch
    w = I.config1(ng=(8, 4), T=1.0)
    f = lcs.Field.from_workload(w)
    sd = torch.from_numpy(w.seeds()).cuda()
    with pytest.raises(lcs.LcsError):
        lcs.advect_early_cg(f, w.ng, w.seed_spacing, w.seed_periodic, w.period, sd, w.t0, w.tf, w.h, 0)
    out = lcs.advect_early_cg(f, w.ng, w.seed_spacing, w.seed_periodic, w.period, sd, w.t0, w.tf, w.h, 3)
    F0, fl0, es0 = f.advect(sd, w.t0, w.tf, w.h)
    cg0, ft0, st0 = lcs.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, F0, fl0, w.tf - w.t0)
    torch.cuda.synchronize()
    assert torch.equal(out[0], F0) and torch.equal(out[4], ft0) and torch.equal(out[3], cg0) and torch.equal(out[6], st0)
    assert float(out[5].min()) == w.tf - w.t0


# -------------------------------------------------------------------------------------------------
# row f4 (first part): Gaussian smoothing of the FTLE field
@pytest.mark.parametrize("dt", [np.float64, np.float32])
def test_smooth_gaussian_vs_oracle(lcs, oracle, dt):
    """lcs_smooth_gaussian against oracle rule O11 on (i) the FTLE field of config 1 reduced with undefined (NaN) seeds punched
    in, non-periodic 2D, and (ii) the FTLE field of config 3 reduced, periodic 3D; ragged sizes, two sigmas."""
    import torch
    tol = 1e-13 if dt == np.float64 else 2e-6
    w = I.config1(ng=(70, 37), T=4.0)
    f, sd, F, flag, es = gpu_run(w)
    flag = flag.clone(); flag[::53] = 1
    _, ft, _ = gpu_cg(w, F, flag)
    w3 = I.config3(ngrid=22, nn=16, T=1.0, n_snap=4)
    f3, sd3, F3, flag3, es3 = gpu_run(w3)
    _, ft3, _ = gpu_cg(w3, F3, flag3)
    for (dim, ng, per, field) in ((2, w.ng, w.seed_periodic, ft), (3, w3.ng, w3.seed_periodic, ft3)):
        field = field.to(torch.float64 if dt == np.float64 else torch.float32).contiguous()
        for sigma in (0.8, 2.5):
            out = cpu(lcs.smooth_gaussian(dim, ng, per, sigma, field)).astype(np.float64)
            ref = oracle.smooth_gaussian(dim, ng[:dim], per[:dim], sigma, cpu(field).astype(np.float64))
            assert np.array_equal(np.isnan(out), np.isnan(ref))
            ok = np.isfinite(ref)
            assert ok.sum() > 1000 and np.max(np.abs(out[ok] - ref[ok])) <= tol * max(1.0, np.abs(ref[ok]).max())
    assert np.isnan(cpu(ft)).sum() > 10
    with pytest.raises(lcs.LcsError):
        lcs.smooth_gaussian(2, w.ng, w.seed_periodic, 0.0, ft)
    with pytest.raises(lcs.LcsError):
        lcs.smooth_gaussian(2, w.ng, w.seed_periodic, 30.0, ft)


# -------------------------------------------------------------------------------------------------
# row f4 (second part): Adams-Bashforth 4 integrator
@pytest.mark.parametrize("case", ["cart2_f64", "cart3_f32_periodic", "tri_f64", "tet_f32", "cart2_f64_exits"])
def test_adams_bashforth_vs_oracle(lcs, oracle, case):
    """integrator = 3 (AB4 with RK4 start-up) against oracle rule O12 on every mesh kind: fp64 cases within the fp64 gate
    (flags and exit steps identical), fp32 cases within the statistical gate.  Windows of several launches exercise the
    velocity history that is carried across launches."""
    if case == "cart2_f64":
        w = I.config1(ng=(64, 32), T=6.0)
    elif case == "cart3_f32_periodic":
        w = I.config3(ngrid=24, nn=16, T=2.0, h=0.01, n_snap=9)
    elif case == "tri_f64":
        w = I.config2(ng=(64, 32), lattice=(50, 25), T=4.0)
    elif case == "tet_f32":
        w = I.config4(ng=(16, 16, 24), delta=0.08, T=1.5, h=0.005, n_snap=10, length=4.0)
    else:
        A = np.array([[0.25, 0.6], [-0.6, 0.25]])
        w = I.analytic_cartesian(2, I.linear_flow(A), (41, 41), (-2.0, -2.0), (0.1, 0.1), (0.0, 2.0, 4.0), ng=(24, 20), seed_lo=(-2.1, -1.4),
                                 seed_spacing=(0.175, 0.14), t0=0.0, tf=4.0, h=0.05)
    fo = oracle.OracleField.from_workload(w)
    Fo, flo, eso = fo.advect_ab4(w.seeds().astype(np.float64), w.t0, w.tf, w.h)
    f, sd, F, flag, es = gpu_run(w, options=dict(integrator=3))
    cgo, fto, sto = oracle_cg(oracle, w, Fo, flo)
    cgg, ftg, stg = gpu_cg(w, F, flag)
    if w.compute_dtype == np.float64 and case != "tri_f64":
        gate_fp64(cpu(F), Fo, cpu(ftg), fto, w.tf - w.t0, cpu(flag), flo, cpu(es), eso)
    elif case == "tri_f64":
        assert np.array_equal(cpu(flag), flo) and np.max(np.abs(cpu(F) - Fo)) <= 1e-10
    else:
        gate_statistical(cpu(F), Fo, cpu(ftg), fto, w.L, cpu(flag), flo)
    if case == "cart2_f64_exits":
        assert set(np.unique(flo)) == {0, 1, 2}
    # and it is a different scheme from RK4: the two flow maps differ by the truncation error, not by rounding
    f2, sd2, F2, flag2, es2 = gpu_run(w)
    both = (cpu(flag) == 0) & (cpu(flag2) == 0)
    d = np.max(np.abs(cpu(F)[both].astype(np.float64) - cpu(F2)[both].astype(np.float64)))
    assert d > (1e-9 if w.compute_dtype == np.float64 else 0.0)


# -------------------------------------------------------------------------------------------------
# randomized small Cartesian configurations: every integrator variant against the oracle
def test_random_cartesian_configs_all_variants(lcs, oracle):
    """24 seeded random small workloads: 2D / 3D, ragged non-power-of-two grids, any mix of periodic axes, fp64 or fp32,
    forward or backward time, step sizes that do or do not divide the snapshot spacing, seeds partly outside.  Each runs
    through a random integrator variant (fused, split, bundled, pre-blended, Adams-Bashforth) and is compared with the oracle:
    fp64 to 1e-9 with identical flags and exit steps, fp32 statistically."""
    rng = np.random.default_rng(777)
    n_exit_cases = 0
    for case in range(24):
        dim = int(rng.integers(2, 4))
        n = tuple(int(v) for v in rng.integers(5, 20, dim))
        per = tuple(int(v) for v in rng.integers(0, 2, dim))
        f32 = bool(rng.integers(0, 2))
        spacing = tuple(float(v) for v in rng.uniform(0.05, 0.2, dim))
        origin = tuple(float(v) for v in rng.uniform(-1, 1, dim))
        ext = [spacing[a] * (n[a] if per[a] else n[a] - 1) for a in range(dim)]
        A = rng.uniform(-0.4, 0.4, (dim, dim))
        b = rng.uniform(-0.3, 0.3, dim)
        times = np.arange(0.0, 2.01, 0.5)
        h = float(rng.choice([0.05, 0.0625, 0.03]))
        nsteps = int(rng.integers(8, 30))
        backward = bool(rng.integers(0, 2))
        t0 = 2.0 if backward else 0.0
        tf = t0 + (-h if backward else h) * nsteps
        ng = tuple(int(v) for v in rng.integers(6, 14, dim))
        margin = 0.0 if all(per) else 0.08
        seed_lo = tuple(origin[a] - margin * ext[a] for a in range(dim))
        seed_sp = tuple((1 + 2 * margin) * ext[a] / ng[a] for a in range(dim))
        dt = np.float32 if f32 else np.float64
        w = I.analytic_cartesian(dim, I.linear_flow(A, b), n, origin, spacing, times, ng=ng, seed_lo=seed_lo, seed_spacing=seed_sp,
                                 t0=t0, tf=tf, h=(-h if backward else h), periodic=per + (0,) * (3 - dim), seed_periodic=(0, 0, 0),
                                 vel_dtype=dt, compute_dtype=dt)
        variant = [dict(bundle=0), dict(bundle=1, bundle_steps=int(rng.integers(1, 9))), dict(integrator=2, bundle=int(rng.integers(0, 2))),
                   dict(bundle=1, preblend=1, preblend_steps=int(rng.integers(1, 9))), dict(integrator=3),
                   dict(bundle=1, bundle_order=0, ld256=0)][case % 6]
        fo = oracle.OracleField.from_workload(w)
        s64 = w.seeds().astype(np.float64)
        if variant.get("integrator") == 3:
            Fo, flo, eso = fo.advect_ab4(s64, w.t0, w.tf, w.h)
        else:
            Fo, flo, eso = fo.advect(s64, w.t0, w.tf, w.h)
        f, sd, F, flag, es = gpu_run(w, options=variant)
        Fg, fg, eg = cpu(F).astype(np.float64), cpu(flag), cpu(es)
        n_exit_cases += int((flo == 1).any())
        tag = "case %d dim %d n %s per %s f32 %s variant %s" % (case, dim, n, per, f32, variant)
        if not f32:
            assert np.array_equal(fg, flo) and np.array_equal(eg, eso), tag
            assert np.max(np.abs(Fg - Fo)) <= 1e-9, tag
        else:
            same = (fg == flo)
            assert same.mean() >= 0.98, tag
            assert np.max(np.linalg.norm(Fg[same] - Fo[same], axis=1)) <= 2e-4 * max(ext), tag
    assert n_exit_cases >= 8


def test_random_simplex_configs_all_variants(lcs, oracle):
    """12 seeded random small simplicial workloads (jittered Delaunay triangles / tets, randomly permuted cell order and vertex
    order within cells so that orientation and local face numbering are arbitrary), fp64 or fp32, forward or backward, through the
    unbundled, bundled, Adams-Bashforth and split per-stage variants.  lcs_locate is bit-exact against brute force on every seed; interior results
    match to 1e-9 (fp64) where both sides agree on the exit flag, and flags agree on >= 98% of the seeds (the in-loop walk uses a
    tolerance at hull faces)."""
    import torch
    rng = np.random.default_rng(4242)
    for case in range(12):
        dim = 2 + case % 2
        if dim == 2:
            V, Cc = I.triangle_mesh_rect(int(rng.integers(8, 16)), int(rng.integers(6, 12)), 2.0, 1.0, rng)
            lo, ext = np.array([0.0, 0.0]), np.array([2.0, 1.0])
        else:
            V, Cc = I.tet_mesh_box(int(rng.integers(5, 8)), rng)
            lo, ext = np.zeros(3), np.ones(3)
        Cc = Cc[rng.permutation(len(Cc))]
        Cc = np.ascontiguousarray(np.stack([c[rng.permutation(dim + 1)] for c in Cc]).astype(np.int32))
        A = rng.uniform(-0.3, 0.3, (dim, dim)); b = rng.uniform(-0.15, 0.15, dim)
        f32 = bool(rng.integers(0, 2)); dt = np.float32 if f32 else np.float64
        backward = bool(rng.integers(0, 2))
        h = 0.05; nsteps = int(rng.integers(10, 30))
        t0 = 2.0 if backward else 0.0
        ng = tuple(int(v) for v in rng.integers(8, 14, dim))
        w = I.analytic_simplex(dim, I.linear_flow(A, b), V, Cc, np.arange(0.0, 2.01, 0.5), ng=ng, seed_lo=tuple(lo - 0.05 * ext),
                               seed_spacing=tuple(1.1 * ext / np.array(ng)), t0=t0, tf=t0 + (-h if backward else h) * nsteps,
                               h=(-h if backward else h), vel_dtype=dt, compute_dtype=dt)
        variant = [dict(bundle=0), dict(bundle=1, bundle_steps=int(rng.integers(1, 9))), dict(integrator=3), dict(integrator=2, bundle=case % 2)][case % 4]
        fo = oracle.OracleField.from_workload(w)
        s64 = w.seeds().astype(np.float64)
        f = lcs.Field.from_workload(w)
        cell = cpu(f.locate(torch.from_numpy(s64).cuda()))
        cb, count = fo.locate_brute(s64)
        tag = "case %d dim %d f32 %s variant %s" % (case, dim, f32, variant)
        assert np.array_equal(cell, cb) and count.max() <= 1, tag
        Fo, flo, eso = (fo.advect_ab4 if variant.get("integrator") == 3 else fo.advect)(s64, w.t0, w.tf, w.h)
        _, sd, F, flag, es = gpu_run(w, options=variant, field=f)
        Fg, fg = cpu(F).astype(np.float64), cpu(flag)
        assert np.array_equal(fg == 2, flo == 2), tag
        same = fg == flo
        assert same.mean() >= 0.98, tag
        eg = cpu(es)
        assert np.all(np.abs(eg[same] - eso[same]) <= 1), tag               # a hull exit may be seen one step apart (walk tolerance)
        exact = same & (eg == eso)
        assert exact.mean() >= 0.97, tag
        assert np.max(np.linalg.norm(Fg[exact] - Fo[exact], axis=1)) <= (2e-4 if f32 else 1e-9), tag
        assert f.info("locate_fallbacks") == 0, tag


# -------------------------------------------------------------------------------------------------
# row f4 (third part): ridge indicator of the smoothed FTLE field
@pytest.mark.parametrize("dt", [np.float64, np.float32])
def test_ridge_vs_oracle(lcs, oracle, dt):
    """lcs_ridge against oracle rule O13 on the smoothed FTLE fields of config 1 (2D, non-periodic, with undefined seeds) and
    config 3 (3D, periodic), both produced by the GPU path, and on an analytic ring.  kappa and d within tolerance; the mask is
    an integer decided by fp64 comparisons on both sides: it must be identical wherever none of the three comparisons is within
    the tolerance of its threshold."""
    import torch
    tol = 1e-9 if dt == np.float64 else 2e-5     # fp32 field values differenced over dx^2: 4 x 1e-7 s / dx^2 relative to max |kappa|
    tdt = torch.float64 if dt == np.float64 else torch.float32
    w = I.config1(ng=(96, 48), T=8.0)
    f, sd, F, flag, es = gpu_run(w)
    flag = flag.clone(); flag[::211] = 1
    _, ft, _ = gpu_cg(w, F, flag)
    s1 = lcs.smooth_gaussian(2, w.ng, w.seed_periodic, 1.5, ft.to(tdt).contiguous())
    w3 = I.config3(ngrid=24, nn=16, T=2.0, n_snap=6)
    f3, sd3, F3, flag3, es3 = gpu_run(w3)
    _, ft3, _ = gpu_cg(w3, F3, flag3)
    s3 = lcs.smooth_gaussian(3, w3.ng, w3.seed_periodic, 1.0, ft3.to(tdt).contiguous())
    n2 = 81
    Xc, Yc = np.meshgrid((np.arange(n2) - 40) * 0.05, (np.arange(n2) - 40) * 0.05)
    ring = torch.from_numpy(np.exp(-(np.hypot(Xc, Yc) - 1.2) ** 2 / (2 * 0.25 ** 2)).ravel().astype(dt)).cuda()
    n_masked = 0
    for (dim, ng, dx, per, field, kmin, smin) in ((2, w.ng, w.seed_spacing, w.seed_periodic, s1, 0.0, 0.05),
                                                   (3, w3.ng, w3.seed_spacing, w3.seed_periodic, s3, 0.0, 0.1),
                                                   (2, (n2, n2, 1), (0.05, 0.05, 1.0), (0, 0, 0), ring, 1.0, 0.8)):
        kap, d, m = (cpu(t) for t in lcs.ridge(dim, ng, dx, per, kmin, smin, field))
        ko, do, mo = oracle.ridge(dim, ng[:dim], dx[:dim], per[:dim], kmin, smin, cpu(field).astype(np.float64))
        assert np.array_equal(np.isnan(kap), np.isnan(ko))
        ok = np.isfinite(ko)
        scale = max(1.0, np.abs(ko[ok]).max())
        assert ok.sum() > 1000 and np.max(np.abs(kap[ok] - ko[ok])) <= tol * scale and np.max(np.abs(d[ok] - do[ok])) <= tol * scale
        delta = min(dx[:dim])
        sv = cpu(field).astype(np.float64)
        margin = np.minimum(np.abs(ko + kmin), np.abs(np.abs(do) - np.abs(ko) * delta / 2))
        clear = ok & (margin > 10 * tol * scale) & (np.abs(sv - smin) > 1e-6)
        assert clear.sum() > 0.5 * ok.sum(), (clear.sum(), ok.sum(), scale)     # the flat far field of the ring sits at the thresholds
        assert np.array_equal(m[clear], mo[clear]) and np.all(m[~ok] == 0)
        n_masked += int(mo.sum())
    assert n_masked > 300
