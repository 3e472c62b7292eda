"""ctypes wrapper of the CPU oracle (oracle/lcs_oracle.c).  TEST INFRASTRUCTURE ONLY.

Allowed users of this module: tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs, nothing else.  The CUDA binding (paper_2209_13775_b200.lcs) is never loaded
from here and no code is shared with it.  Argument marshalling only: the arithmetic is in lcs_oracle.c, with one exception:
the update rule of oracle rule O10 (early Cauchy-Green evaluation: which seeds are re-evaluated at an evaluation point and which
keep their last result) is the numpy mask bookkeeping of `advect_early_cg` below, written from DESIGN.md reading #29; every
evaluation it triggers is the C routine orc_cg_ftle.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lcs_oracle.c")
_LIB = os.path.join(_HERE, "liblcs_oracle.so")


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no FMA contraction, OpenMP over seeds)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Field(C.Structure):
    _fields_ = [("dim", C.c_int32), ("kind", C.c_int32),
                ("n", C.c_int32 * 3), ("periodic", C.c_int32 * 3),
                ("origin", C.c_double * 3), ("spacing", C.c_double * 3),
                ("nv", C.c_int64), ("nc", C.c_int64),
                ("verts", C.c_void_p), ("cells", C.c_void_p), ("neigh", C.c_void_p),
                ("ns", C.c_int32), ("vel_f32", C.c_int32),
                ("times", C.c_void_p), ("vel", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_eigmax_sym2.restype = C.c_double
        _lib.orc_eigmax_sym2.argtypes = [C.c_double] * 3
        _lib.orc_eigmax_sym3.restype = C.c_double
        _lib.orc_eigmax_sym3.argtypes = [C.c_double] * 6
        _lib.orc_simplex_build_neighbours.restype = C.c_int
        _lib.orc_max_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleField:
    """Field description for the oracle.  Keeps numpy arrays alive; builds the face-neighbour table
    of a simplex mesh with the oracle's own routine."""

    def __init__(self, dim, kind, times, vel, n=(1, 1, 1), origin=(0, 0, 0), spacing=(1, 1, 1),
                 periodic=(0, 0, 0), vertices=None, cells=None):
        self.dim, self.kind = int(dim), int(kind)
        self.times = np.ascontiguousarray(times, dtype=np.float64)
        assert vel.dtype in (np.float32, np.float64)
        self.vel = np.ascontiguousarray(vel)
        self.verts = None if vertices is None else np.ascontiguousarray(vertices, dtype=np.float64)
        self.cells = None if cells is None else np.ascontiguousarray(cells, dtype=np.int32)
        self.neigh = None
        f = _Field()
        f.dim, f.kind = self.dim, self.kind
        for a in range(3):
            f.n[a] = int(n[a]) if a < len(n) else 1
            f.periodic[a] = int(periodic[a]) if a < len(periodic) else 0
            f.origin[a] = float(origin[a]) if a < len(origin) else 0.0
            f.spacing[a] = float(spacing[a]) if a < len(spacing) else 1.0
        if self.kind == 1:
            f.nv, f.nc = self.verts.shape[0], self.cells.shape[0]
            self.neigh = np.empty_like(self.cells)
            rc = lib().orc_simplex_build_neighbours(C.c_int32(self.dim), C.c_int64(f.nc),
                                                    _p(self.cells), _p(self.neigh))
            if rc != 0:
                raise ValueError("mesh error %d" % rc)
            assert self.vel.shape[1] == f.nv
        else:
            f.nv = f.n[0] * f.n[1] * f.n[2]
            assert self.vel.shape[1] == f.nv, (self.vel.shape, f.nv)
        f.verts, f.cells, f.neigh = _p(self.verts), _p(self.cells), _p(self.neigh)
        f.ns = len(self.times)
        f.vel_f32 = 1 if self.vel.dtype == np.float32 else 0
        f.times, f.vel = _p(self.times), _p(self.vel)
        self._f = f

    @classmethod
    def from_workload(cls, w):
        return cls(w.dim, w.kind, w.times, w.vel, n=w.n, origin=w.origin, spacing=w.spacing,
                   periodic=w.periodic, vertices=w.vertices, cells=w.cells)

    # ---- location ---------------------------------------------------------------------------
    def cart_locate(self, pos):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        n = pos.shape[0]
        cell = np.empty(n, dtype=np.int32)
        w = np.zeros((n, self.dim), dtype=np.float64)
        lib().orc_cart_locate(C.byref(self._f), C.c_int64(n), _p(pos), _p(cell), _p(w))
        return cell, w

    def locate_brute(self, pos):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        n = pos.shape[0]
        cell = np.empty(n, dtype=np.int32)
        count = np.empty(n, dtype=np.int32)
        lib().orc_simplex_locate_brute(C.byref(self._f), C.c_int64(n), _p(pos), _p(cell), _p(count))
        return cell, count

    def accepts(self, pos, cell):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        cell = np.ascontiguousarray(cell, dtype=np.int32)
        ok = np.empty(pos.shape[0], dtype=np.int32)
        lib().orc_simplex_accepts(C.byref(self._f), C.c_int64(pos.shape[0]), _p(pos), _p(cell), _p(ok))
        return ok.astype(bool)

    def locate_walk(self, pos, start=None):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        n = pos.shape[0]
        if start is None:
            start = self.start_hint(pos)
        start = np.ascontiguousarray(start, dtype=np.int32)
        cell = np.empty(n, dtype=np.int32)
        lib().orc_simplex_locate_walk(C.byref(self._f), C.c_int64(n), _p(pos), _p(start), _p(cell))
        return cell

    def start_hint(self, pos):
        """A start cell for the walk: any cell incident on the nearest mesh vertex (scipy cKDTree, a
        library primitive).  The walk's result does not depend on it (canonical predicate => unique)."""
        from scipy.spatial import cKDTree
        if not hasattr(self, "_tree"):
            self._tree = cKDTree(self.verts)
            v2c = np.zeros(self.verts.shape[0], dtype=np.int32)
            ids = np.repeat(np.arange(self.cells.shape[0], dtype=np.int32), self.dim + 1)
            v2c[self.cells.ravel()] = ids
            self._v2c = v2c
        _, nearest = self._tree.query(np.asarray(pos, dtype=np.float64), workers=-1)
        return self._v2c[nearest]

    def locate(self, pos):
        """-1 = outside.  Cartesian: O2 formula; simplex: canonical-predicate walk (fast mode)."""
        if self.kind == 0:
            return self.cart_locate(pos)[0]
        return self.locate_walk(pos)

    # ---- interpolation ----------------------------------------------------------------------
    def velocity(self, pos, t, start=None):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        n = pos.shape[0]
        if self.kind == 1 and start is None:
            start = self.start_hint(pos)
        st = None if start is None else np.ascontiguousarray(start, dtype=np.int32)
        u = np.empty((n, self.dim), dtype=np.float64)
        inside = np.empty(n, dtype=np.int32)
        lib().orc_velocity(C.byref(self._f), C.c_int64(n), _p(pos), C.c_double(t), _p(st), _p(u), _p(inside))
        return u, inside.astype(bool)

    # ---- RK4 flow map -----------------------------------------------------------------------
    def advect(self, seeds, t0, tf, h, rec_every=0):
        seeds = np.ascontiguousarray(seeds, dtype=np.float64)      # fp32 seeds are widened exactly
        n = seeds.shape[0]
        cell0 = self.locate_walk(seeds) if self.kind == 1 else None
        F = np.empty_like(seeds)
        flag = np.empty(n, dtype=np.uint8)
        es = np.empty(n, dtype=np.int32)
        traj = None
        if rec_every > 0:
            N = int(round((tf - t0) / h))
            traj = np.empty((N // rec_every, n, self.dim), dtype=np.float64)
        lib().orc_advect(C.byref(self._f), C.c_int64(n), _p(seeds), C.c_double(t0), C.c_double(tf),
                         C.c_double(h), _p(cell0), _p(F), _p(flag), _p(es), C.c_int32(rec_every), _p(traj))
        if rec_every > 0:
            return F, flag, es, traj
        return F, flag, es

    def advect_ab4(self, seeds, t0, tf, h):
        """Rule O12: 4-step Adams-Bashforth with an RK4 start-up."""
        seeds = np.ascontiguousarray(seeds, dtype=np.float64)
        n = seeds.shape[0]
        cell0 = self.locate_walk(seeds) if self.kind == 1 else None
        F = np.empty_like(seeds)
        flag = np.empty(n, dtype=np.uint8)
        es = np.empty(n, dtype=np.int32)
        lib().orc_advect_ab4(C.byref(self._f), C.c_int64(n), _p(seeds), C.c_double(t0), C.c_double(tf), C.c_double(h), _p(cell0),
                             _p(F), _p(flag), _p(es))
        return F, flag, es


def cg_ftle(dim, ng, seed_spacing, seed_periodic, period, flowmap, exit_flag, T):
    """Returns (cg [n][3|6], ftle [n], status [n])."""
    F = np.ascontiguousarray(flowmap, dtype=np.float64)
    n = F.shape[0]
    ng_ = np.asarray(list(ng) + [1] * (3 - len(ng)), dtype=np.int32)
    dx = np.asarray(list(seed_spacing) + [1.0] * (3 - len(seed_spacing)), dtype=np.float64)
    sp = np.asarray(list(seed_periodic) + [0] * (3 - len(seed_periodic)), dtype=np.int32)
    per = np.asarray(list(period) + [0.0] * (3 - len(period)), dtype=np.float64)
    assert n == int(ng_[0]) * int(ng_[1]) * (int(ng_[2]) if dim == 3 else 1)
    fl = None if exit_flag is None else np.ascontiguousarray(exit_flag, dtype=np.uint8)
    cg = np.empty((n, 3 if dim == 2 else 6), dtype=np.float64)
    ftle = np.empty(n, dtype=np.float64)
    status = np.empty(n, dtype=np.uint8)
    lib().orc_cg_ftle(C.c_int32(dim), _p(ng_), _p(dx), _p(sp), _p(per), _p(F), _p(fl), C.c_double(T),
                      _p(cg), _p(ftle), _p(status))
    return cg, ftle, status


def early_cg(field, dim, ng, seed_spacing, seed_periodic, period, seeds, t0, tf, h, every):
    """Rule O10 (row f1, reading #29): early evaluation of the Cauchy-Green tensor when a stencil member leaves.
    All tracers advance synchronously (positions of all tracers exist at every step, so C "can be evaluated
    at any time step"); when a tracer leaves the domain, "the computation of the CG tensor is performed" for the stencils it
    belongs to with the positions at that time instead of discarding them.
    Evaluation points are the step counts m = every, 2 every, ... and N.  At m a tracer is alive if it has completed m steps.
    Seed i is (re-)evaluated at m iff it is alive and each of its 2 dim grid neighbours is alive or never started (flag 2 / outside
    the grid: those are invalid neighbours in the sense of O5, i.e. one-sided differences); a neighbour that left freezes
    the seed at its previous evaluation.  The evaluation is O5-O7 with T_eff = m h.  Returns
    (flowmap, flag, exit_step, cg, ftle, t_eff, status); seeds never evaluated have NaN, t_eff = 0 and status bit 0."""
    n = seeds.shape[0]
    N = int(round((tf - t0) / h))
    assert every >= 1
    F, flag, es, traj = field.advect(seeds, t0, tf, h, rec_every=every)
    ncg = 3 if dim == 2 else 6
    cg = np.full((n, ncg), np.nan)
    ftle = np.full(n, np.nan)
    t_eff = np.zeros(n)
    status = np.ones(n, dtype=np.uint8)
    g = [int(ng[a]) if a < dim else 1 for a in range(3)]
    idx = np.arange(n).reshape(g[2], g[1], g[0])
    points = [(m, traj[m // every - 1]) for m in range(every, N + 1, every)]
    if N % every != 0:
        points.append((N, F))
    for m, Fm in points:
        alive = (flag == 0) | ((flag == 1) & (es >= m))
        left = (flag == 1) & (es < m)
        never = (flag == 2)
        update = alive.copy()
        for a in range(dim):
            ax = 2 - a                                           # axis 0 is the fastest index
            for sh in (1, -1):
                nb = np.roll(idx, -sh, axis=ax)
                nb_left = left[nb]
                if not seed_periodic[a]:                         # outside the grid: no neighbour, never blocks
                    sl = [slice(None)] * 3
                    sl[ax] = -1 if sh == 1 else 0
                    nb_left = nb_left.copy()
                    nb_left[tuple(sl)] = False
                update &= ~nb_left.ravel()
        cgm, ftm, stm = cg_ftle(dim, ng, seed_spacing, seed_periodic, period, Fm, (never | left).astype(np.uint8), m * h)
        cg[update] = cgm[update]
        ftle[update] = ftm[update]
        status[update] = stm[update]
        t_eff[update] = m * h
    return F, flag, es, cg, ftle, t_eff, status


def cg_ftle_aux(dim, delta, flow_aux, flag_aux, T):
    """Rule O9.  flow_aux [n][2 dim][dim] (entry 2b: released at +delta_b, 2b+1: at -delta_b), flag_aux [n][2 dim] or None.
    Returns (cg, ftle, status)."""
    Fa = np.ascontiguousarray(flow_aux, dtype=np.float64).reshape(-1, 2 * dim, dim)
    n = Fa.shape[0]
    dl = np.ascontiguousarray(delta, dtype=np.float64)
    fl = None if flag_aux is None else np.ascontiguousarray(flag_aux, dtype=np.uint8).reshape(n, 2 * dim)
    cg = np.empty((n, 3 if dim == 2 else 6), dtype=np.float64)
    ftle = np.empty(n, dtype=np.float64)
    status = np.empty(n, dtype=np.uint8)
    lib().orc_cg_ftle_aux(C.c_int32(dim), C.c_int64(n), _p(dl), _p(Fa), _p(fl), C.c_double(T), _p(cg), _p(ftle), _p(status))
    return cg, ftle, status


def smooth_gaussian(dim, ng, seed_periodic, sigma, field):
    """Rule O11: NaN-aware normalised Gaussian smoothing of a scalar field on the seed grid, one pass per axis."""
    f = np.ascontiguousarray(field, dtype=np.float64).ravel()
    ng_ = np.asarray(list(ng) + [1] * (3 - len(ng)), dtype=np.int32)
    sp = np.asarray(list(seed_periodic) + [0] * (3 - len(seed_periodic)), dtype=np.int32)
    out = np.empty_like(f)
    lib().orc_smooth_gaussian(C.c_int32(dim), _p(ng_), _p(sp), C.c_double(sigma), _p(f), _p(out))
    return out


def ridge(dim, ng, seed_spacing, seed_periodic, kappa_min, s_min, field):
    """Rule O13: second-derivative ridge indicator of a scalar field on the seed grid.  Returns (kappa, d, mask)."""
    f = np.ascontiguousarray(field, dtype=np.float64).ravel()
    ng_ = np.asarray(list(ng) + [1] * (3 - len(ng)), dtype=np.int32)
    dx = np.asarray(list(seed_spacing) + [1.0] * (3 - len(seed_spacing)), dtype=np.float64)
    sp = np.asarray(list(seed_periodic) + [0] * (3 - len(seed_periodic)), dtype=np.int32)
    kappa, d, mask = np.empty_like(f), np.empty_like(f), np.empty(f.size, dtype=np.uint8)
    lib().orc_ridge(C.c_int32(dim), _p(ng_), _p(dx), _p(sp), C.c_double(kappa_min), C.c_double(s_min), _p(f), _p(kappa), _p(d), _p(mask))
    return kappa, d, mask


def cg_eigen(dim, cg):
    """All eigenvalues (ascending) and unit eigenvectors (row i belongs to eigenvalue i) of C: rule O8."""
    c = np.ascontiguousarray(cg, dtype=np.float64)
    n = c.shape[0]
    assert c.shape[1] == (3 if dim == 2 else 6)
    evals = np.empty((n, dim), dtype=np.float64)
    evecs = np.empty((n, dim, dim), dtype=np.float64)
    lib().orc_cg_eigen(C.c_int32(dim), C.c_int64(n), _p(c), _p(evals), _p(evecs))
    return evals, evecs


def eigmax_sym2(c11, c12, c22):
    return lib().orc_eigmax_sym2(c11, c12, c22)


def eigmax_sym3(c11, c12, c13, c22, c23, c33):
    return lib().orc_eigmax_sym3(c11, c12, c13, c22, c23, c33)


def max_threads():
    return int(lib().orc_max_threads())
