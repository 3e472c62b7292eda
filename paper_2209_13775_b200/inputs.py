"""Seeded synthetic inputs for the LCS hot path (fields, meshes, seed grids).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic: no cell search, no interpolation, no RK4, no
finite differences, no eigenvalues.  It only samples analytic velocity fields
on mesh nodes, builds meshes and lays out seed grids.  It imports neither
``oracle/`` nor the CUDA binding.

The five workloads stand in for the paper's datasets (double gyre, Rayleigh-
Benard cell, coronary stenosis, AAA), which are not available:
same structure (2D/3D x Cartesian/unstructured, fp64/fp32, 1e5..1e7 elements
and seeds), recipes from BASELINE.json `configs` and
SURVEY.md section 8.3.  RNG: numpy default_rng(2209137750 + config number).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional, Sequence

import numpy as np

SEED_BASE = 2209137750

CARTESIAN = 0
SIMPLEX = 1


# ----------------------------------------------------------------------------
# analytic velocity fields (input data, evaluated on mesh nodes only)
# ----------------------------------------------------------------------------
def double_gyre(p: np.ndarray, t: float, A=0.1, eps=0.25, omega=2 * np.pi / 10) -> np.ndarray:
    """Double gyre of the paper's ref [29]; psi = A sin(pi f) sin(pi y),
    f = a(t) x^2 + b(t) x, a = eps sin(omega t), b = 1 - 2 a; u = -dpsi/dy, v = dpsi/dx."""
    x, y = p[:, 0], p[:, 1]
    a = eps * np.sin(omega * t)
    b = 1.0 - 2.0 * a
    f = a * x * x + b * x
    dfdx = 2.0 * a * x + b
    u = -np.pi * A * np.sin(np.pi * f) * np.cos(np.pi * y)
    v = np.pi * A * np.cos(np.pi * f) * np.sin(np.pi * y) * dfdx
    return np.stack([u, v], axis=1)


def abc_flow(p: np.ndarray, t: float) -> np.ndarray:
    """Time-dependent ABC flow of BASELINE.json configs 3/5."""
    x, y, z = p[:, 0], p[:, 1], p[:, 2]
    A = np.sqrt(3.0) * (1.0 + 0.1 * np.sin(np.pi * t))
    B = np.sqrt(2.0)
    C = 1.0
    return np.stack([A * np.sin(z) + C * np.cos(y),
                     B * np.sin(x) + A * np.cos(z),
                     C * np.sin(y) + B * np.cos(x)], axis=1)


def pipe_flow(p: np.ndarray, t: float) -> np.ndarray:
    """Poiseuille 2(1-r^2) axial + swirl 0.2 sin(2 pi t/5) sin(pi z/5) (-y, x) (config 4)."""
    x, y, z = p[:, 0], p[:, 1], p[:, 2]
    s = 0.2 * np.sin(2 * np.pi * t / 5.0) * np.sin(np.pi * z / 5.0)
    return np.stack([-s * y, s * x, 2.0 * (1.0 - (x * x + y * y))], axis=1)


def linear_flow(A: np.ndarray, b: Optional[np.ndarray] = None) -> Callable:
    """u = A x + b (steady); used by the closed-form pins P1-P7."""
    A = np.asarray(A, dtype=np.float64)
    bb = np.zeros(A.shape[0]) if b is None else np.asarray(b, dtype=np.float64)
    return lambda p, t: p @ A.T + bb


def time_linear_uniform(a: Sequence[float], b: Sequence[float]) -> Callable:
    """u = a + b t, uniform in space (pin P8)."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return lambda p, t: np.broadcast_to(a + b * t, p.shape).copy()


# ----------------------------------------------------------------------------
# workload container
# ----------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    dim: int
    kind: int                                  # CARTESIAN | SIMPLEX
    times: np.ndarray                          # [ns] fp64, uniform
    vel: np.ndarray                            # [ns][nv][dim], fp32 or fp64
    compute_dtype: np.dtype                    # positions / arithmetic inside advect
    # Cartesian description
    n: tuple = (1, 1, 1)                       # nodes per axis
    origin: tuple = (0.0, 0.0, 0.0)
    spacing: tuple = (1.0, 1.0, 1.0)
    periodic: tuple = (0, 0, 0)
    # simplex description
    vertices: Optional[np.ndarray] = None      # [nv][dim] fp64
    cells: Optional[np.ndarray] = None         # [nc][dim+1] int32, any orientation
    # seeds (structured grid, axis 0 fastest)
    ng: tuple = (1, 1, 1)
    seed_lo: tuple = (0.0, 0.0, 0.0)
    seed_spacing: tuple = (1.0, 1.0, 1.0)
    seed_periodic: tuple = (0, 0, 0)
    period: tuple = (0.0, 0.0, 0.0)
    t0: float = 0.0
    tf: float = 1.0
    h: float = 0.1
    L: float = 1.0                             # domain length used by the fp32 gate
    meta: dict = field(default_factory=dict)

    @property
    def n_seeds(self) -> int:
        return int(self.ng[0]) * int(self.ng[1]) * int(self.ng[2])

    @property
    def n_steps(self) -> int:
        return int(round((self.tf - self.t0) / self.h))

    def seeds(self, dtype=None) -> np.ndarray:
        """Cell-centred seed grid [n][dim], axis 0 fastest (SURVEY reading #23)."""
        return seed_grid(self.dim, self.ng, self.seed_lo, self.seed_spacing,
                         dtype or self.compute_dtype)

    def nodes(self) -> np.ndarray:
        if self.kind == SIMPLEX:
            return self.vertices
        return cartesian_nodes(self.dim, self.n, self.origin, self.spacing)


def seed_grid(dim, ng, lo, spacing, dtype=np.float64) -> np.ndarray:
    """x_i = lo + (i + 1/2) * spacing, computed in fp64 then cast; index = i0 + ng0*(i1 + ng1*i2)."""
    axes = [np.float64(lo[a]) + (np.arange(ng[a], dtype=np.float64) + 0.5) * np.float64(spacing[a])
            for a in range(dim)]
    if dim == 2:
        Y, X = np.meshgrid(axes[1], axes[0], indexing="ij")
        out = np.stack([X.ravel(), Y.ravel()], axis=1)
    else:
        Z, Y, X = np.meshgrid(axes[2], axes[1], axes[0], indexing="ij")
        out = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    return np.ascontiguousarray(out.astype(dtype))


def cartesian_nodes(dim, n, origin, spacing) -> np.ndarray:
    """Node i on axis a at origin[a] + i*spacing[a]; node index = i0 + n0*(i1 + n1*i2)."""
    axes = [np.float64(origin[a]) + np.arange(n[a], dtype=np.float64) * np.float64(spacing[a])
            for a in range(dim)]
    if dim == 2:
        Y, X = np.meshgrid(axes[1], axes[0], indexing="ij")
        return np.stack([X.ravel(), Y.ravel()], axis=1)
    Z, Y, X = np.meshgrid(axes[2], axes[1], axes[0], indexing="ij")
    return np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)


def sample_field(fn: Callable, nodes: np.ndarray, times: np.ndarray, dtype) -> np.ndarray:
    """[ns][nv][dim]: fn evaluated in fp64 on the nodes at each snapshot time, then cast."""
    out = np.empty((len(times), nodes.shape[0], nodes.shape[1]), dtype=dtype)
    for s, t in enumerate(times):
        out[s] = fn(nodes, float(t)).astype(dtype)
    return out


# ----------------------------------------------------------------------------
# meshes
# ----------------------------------------------------------------------------
def triangle_mesh_rect(nx: int, ny: int, lx: float, ly: float, rng: np.random.Generator,
                       jitter: float = 0.35):
    """Jittered-lattice Delaunay triangulation whose hull is exactly [0,lx]x[0,ly]
    (SURVEY 8.3 config 2): interior nodes jittered by U(-j,j)*spacing per axis, boundary
    nodes only tangentially, corners fixed."""
    from scipy.spatial import Delaunay
    hx, hy = lx / (nx - 1), ly / (ny - 1)
    I, J = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    X = I * hx
    Y = J * hy
    jx = rng.uniform(-jitter, jitter, X.shape) * hx
    jy = rng.uniform(-jitter, jitter, Y.shape) * hy
    on_x = (I == 0) | (I == nx - 1)          # on a vertical wall: no x jitter
    on_y = (J == 0) | (J == ny - 1)
    jx[on_x] = 0.0
    jy[on_y] = 0.0
    P = np.stack([(X + jx).ravel(), (Y + jy).ravel()], axis=1)
    # walls exactly on the rectangle
    P[(I == nx - 1).ravel(), 0] = lx
    P[(J == ny - 1).ravel(), 1] = ly
    tri = Delaunay(P)
    return np.ascontiguousarray(P), np.ascontiguousarray(tri.simplices.astype(np.int32))


def tet_mesh_pipe(delta: float, rng: np.random.Generator, radius=1.0, length=10.0, jitter=0.35):
    """Jittered cubic lattice clipped to the cylinder r<=radius, 0<=z<=length, Delaunay
    (no exact wall/cap layers; Qhull output is NOT oriented)."""
    from scipy.spatial import Delaunay
    nx = int(np.ceil(2 * radius / delta)) + 1
    nz = int(np.ceil(length / delta)) + 1
    xs = -radius + np.arange(nx) * delta
    zs = np.arange(nz) * delta
    Z, Y, X = np.meshgrid(zs, xs, xs, indexing="ij")
    P = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    P += rng.uniform(-jitter, jitter, P.shape) * delta
    keep = (np.hypot(P[:, 0], P[:, 1]) <= radius) & (P[:, 2] >= 0.0) & (P[:, 2] <= length)
    P = np.ascontiguousarray(P[keep])
    tet = Delaunay(P)
    return P, np.ascontiguousarray(tet.simplices.astype(np.int32))


def tet_mesh_box(n: int, rng: np.random.Generator, lo=0.0, hi=1.0, jitter=0.3):
    """Small jittered-lattice tet mesh of a cube whose hull is exactly the cube (tests)."""
    from scipy.spatial import Delaunay
    h = (hi - lo) / (n - 1)
    idx = np.arange(n)
    K, J, I = np.meshgrid(idx, idx, idx, indexing="ij")
    P = np.stack([I.ravel(), J.ravel(), K.ravel()], axis=1).astype(np.float64)
    jit = rng.uniform(-jitter, jitter, P.shape)
    on = (P == 0) | (P == n - 1)
    jit[on] = 0.0
    P = lo + (P + jit) * h
    tet = Delaunay(P)
    return np.ascontiguousarray(P), np.ascontiguousarray(tet.simplices.astype(np.int32))


# ----------------------------------------------------------------------------
# the five BASELINE.json configs (each scalable for tests)
# ----------------------------------------------------------------------------
def config1(ng=(256, 128), n_nodes=(201, 101), T=10.0, h=0.1) -> Workload:
    """2D double gyre, Cartesian 201x101 on [0,2]x[0,1], 11 snapshots, fp64."""
    n = (n_nodes[0], n_nodes[1], 1)
    spacing = (2.0 / (n[0] - 1), 1.0 / (n[1] - 1), 1.0)
    times = np.arange(0.0, 10.0 + 0.5, 1.0)
    nodes = cartesian_nodes(2, n, (0, 0, 0), spacing)
    vel = sample_field(double_gyre, nodes, times, np.float64)
    return Workload("cfg1_double_gyre_cart2d_f64", 2, CARTESIAN, times, vel, np.dtype(np.float64),
                    n=n, origin=(0.0, 0.0, 0.0), spacing=spacing, periodic=(0, 0, 0),
                    ng=(ng[0], ng[1], 1), seed_lo=(0.0, 0.0, 0.0),
                    seed_spacing=(2.0 / ng[0], 1.0 / ng[1], 1.0),
                    t0=0.0, tf=T, h=h, L=2.0)


def config2(ng=(1024, 512), lattice=(317, 159), T=15.0, h=0.05) -> Workload:
    """2D double gyre on a Delaunay triangle mesh (50 403 vertices at full size), 31 snapshots, fp64."""
    rng = np.random.default_rng(SEED_BASE + 2)
    V, C = triangle_mesh_rect(lattice[0], lattice[1], 2.0, 1.0, rng)
    times = np.arange(0.0, 15.0 + 0.25, 0.5)
    vel = sample_field(double_gyre, V, times, np.float64)
    return Workload("cfg2_double_gyre_tri_f64", 2, SIMPLEX, times, vel, np.dtype(np.float64),
                    vertices=V, cells=C,
                    ng=(ng[0], ng[1], 1), seed_lo=(0.0, 0.0, 0.0),
                    seed_spacing=(2.0 / ng[0], 1.0 / ng[1], 1.0),
                    t0=0.0, tf=T, h=h, L=2.0)


def _abc_snapshots(nn: int, times: np.ndarray, dtype) -> np.ndarray:
    """ABC field on a periodic nn^3 grid, separable evaluation (fp64 then cast)."""
    x = 2 * np.pi * np.arange(nn, dtype=np.float64) / nn
    sx, cx = np.sin(x), np.cos(x)
    B, C = np.sqrt(2.0), 1.0
    out = np.empty((len(times), nn, nn, nn, 3), dtype=dtype)      # [s][k][j][i][c]
    for s, t in enumerate(times):
        A = np.sqrt(3.0) * (1.0 + 0.1 * np.sin(np.pi * t))
        out[s, ..., 0] = (A * sx[:, None, None] + C * cx[None, :, None])      # A sin z + C cos y
        out[s, ..., 1] = (B * sx[None, None, :] + A * cx[:, None, None])      # B sin x + A cos z
        out[s, ..., 2] = (C * sx[None, :, None] + B * cx[None, None, :])      # C sin y + B cos x
    return out.reshape(len(times), nn ** 3, 3)


def config3(ngrid=256, nn=128, T=5.0, h=0.01, n_snap=21) -> Workload:
    """3D ABC flow, periodic 128^3, 21 snapshots dt=0.5, fp32; 256^3 seeds, 500 steps."""
    times = 0.5 * np.arange(n_snap, dtype=np.float64)
    vel = _abc_snapshots(nn, times, np.float32)
    d = 2 * np.pi / nn
    L = 2 * np.pi
    return Workload("cfg3_abc_cart3d_f32", 3, CARTESIAN, times, vel, np.dtype(np.float32),
                    n=(nn, nn, nn), origin=(0.0, 0.0, 0.0), spacing=(d, d, d), periodic=(1, 1, 1),
                    ng=(ngrid, ngrid, ngrid), seed_lo=(0.0, 0.0, 0.0),
                    seed_spacing=(L / ngrid,) * 3, seed_periodic=(1, 1, 1), period=(L, L, L),
                    t0=0.0, tf=T, h=h, L=L)


def config4(ng=(256, 256, 512), delta=0.025, T=8.0, h=0.005, n_snap=50, length=10.0) -> Workload:
    """3D pipe flow on a Delaunay tet mesh (about 2.0 M vertices / 13.4 M tets at delta=0.025), fp32 data.
    Seeds: bounding-box grid [-1,1]^2 x [0,length], z = pipe axis (SURVEY reading #22)."""
    rng = np.random.default_rng(SEED_BASE + 4)
    V, C = tet_mesh_pipe(delta, rng, 1.0, length)
    times = 0.2 * np.arange(n_snap, dtype=np.float64)
    vel = sample_field(pipe_flow, V, times, np.float32)
    return Workload("cfg4_pipe_tet_f32", 3, SIMPLEX, times, vel, np.dtype(np.float32),
                    vertices=V, cells=C, ng=tuple(ng), seed_lo=(-1.0, -1.0, 0.0),
                    seed_spacing=(2.0 / ng[0], 2.0 / ng[1], length / ng[2]),
                    t0=0.0, tf=T, h=h, L=length)


def config5(ngrid=192, nn=128, n_grids=16, T=5.0, h=0.01, n_snap=41):
    """FTLE time series: config-3 field with 41 snapshots; grid k released at t = 0.5 k + T and
    integrated BACKWARD (h<0) down to t0 = 0.5 k (SURVEY reading #21).  Returns the base workload
    (field + seed grid) and the list of (t_release, t_end) pairs."""
    w = config3(ngrid=ngrid, nn=nn, T=T, h=h, n_snap=n_snap)
    w.name = "cfg5_abc_backward_series_f32"
    windows = [(0.5 * k + T, 0.5 * k) for k in range(n_grids)]
    w.t0, w.tf, w.h = windows[0][0], windows[0][1], -abs(h)
    w.meta["windows"] = windows
    return w


# ----------------------------------------------------------------------------
# small analytic workloads for the closed-form pins and parity edge cases
# ----------------------------------------------------------------------------
def analytic_cartesian(dim, fn, n, origin, spacing, times, ng, seed_lo, seed_spacing, t0, tf, h,
                       periodic=(0, 0, 0), seed_periodic=(0, 0, 0), period=(0.0, 0.0, 0.0),
                       vel_dtype=np.float64, compute_dtype=np.float64, name="analytic_cart") -> Workload:
    n3 = tuple(n) + (1,) * (3 - len(n))
    nodes = cartesian_nodes(dim, n3, tuple(origin) + (0.0,) * (3 - len(origin)),
                            tuple(spacing) + (1.0,) * (3 - len(spacing)))
    times = np.asarray(times, dtype=np.float64)
    vel = sample_field(fn, nodes, times, vel_dtype)
    pad = lambda v, fill: tuple(v) + (fill,) * (3 - len(v))
    return Workload(name, dim, CARTESIAN, times, vel, np.dtype(compute_dtype),
                    n=n3, origin=pad(origin, 0.0), spacing=pad(spacing, 1.0), periodic=pad(periodic, 0),
                    ng=pad(ng, 1), seed_lo=pad(seed_lo, 0.0), seed_spacing=pad(seed_spacing, 1.0),
                    seed_periodic=pad(seed_periodic, 0), period=pad(period, 0.0),
                    t0=t0, tf=tf, h=h, L=float(max(np.asarray(spacing) * (np.asarray(n) - 1))))


def analytic_simplex(dim, fn, vertices, cells, times, ng, seed_lo, seed_spacing, t0, tf, h,
                     vel_dtype=np.float64, compute_dtype=np.float64, name="analytic_simplex") -> Workload:
    times = np.asarray(times, dtype=np.float64)
    vel = sample_field(fn, vertices, times, vel_dtype)
    pad = lambda v, fill: tuple(v) + (fill,) * (3 - len(v))
    ext = vertices.max(axis=0) - vertices.min(axis=0)
    return Workload(name, dim, SIMPLEX, times, vel, np.dtype(compute_dtype),
                    vertices=np.ascontiguousarray(vertices, dtype=np.float64),
                    cells=np.ascontiguousarray(cells, dtype=np.int32),
                    ng=pad(ng, 1), seed_lo=pad(seed_lo, 0.0), seed_spacing=pad(seed_spacing, 1.0),
                    t0=t0, tf=tf, h=h, L=float(ext.max()))


def kuhn_mesh(dim: int, n: int, h: float = 1.0):
    """Structured simplicial mesh of [0,(n-1)h]^dim: every square/cube split into 2/6 Kuhn simplices
    (one per permutation of the axes).  Conforming, exactly representable coordinates for integer h,
    and of mixed orientation (odd permutations are negatively oriented) -- used by the tie-break tests."""
    import itertools
    idx = np.arange(n)
    if dim == 2:
        J, I = np.meshgrid(idx, idx, indexing="ij")
        P = np.stack([I.ravel(), J.ravel()], axis=1).astype(np.float64) * h
        vid = lambda c: c[0] + n * c[1]
    else:
        K, J, I = np.meshgrid(idx, idx, idx, indexing="ij")
        P = np.stack([I.ravel(), J.ravel(), K.ravel()], axis=1).astype(np.float64) * h
        vid = lambda c: c[0] + n * (c[1] + n * c[2])
    cells = []
    for base in itertools.product(range(n - 1), repeat=dim):
        base = base[::-1]
        for perm in itertools.permutations(range(dim)):
            c = list(base)
            vs = [vid(c)]
            for a in perm:
                c[a] += 1
                vs.append(vid(c))
            cells.append(vs)
    return np.ascontiguousarray(P), np.asarray(cells, dtype=np.int32)


def aux_seeds(seeds: np.ndarray, delta: Sequence[float]) -> np.ndarray:
    """Auxiliary points around each seed: [n][2 dim][dim], entry 2b = seed + delta_b e_b, 2b+1 = seed - delta_b e_b
    (layout only; the difference quotient is formed by lcs_cg_ftle_aux / oracle rule O9)."""
    n, dim = seeds.shape
    out = np.repeat(seeds[:, None, :], 2 * dim, axis=1).astype(seeds.dtype)
    for b in range(dim):
        out[:, 2 * b, b] += seeds.dtype.type(delta[b])
        out[:, 2 * b + 1, b] -= seeds.dtype.type(delta[b])
    return out
