"""Thin ctypes binding of liblcs.so (include/lcs.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; torch is used for device memory and
streams.  There is no CPU fallback: importing is cheap, but the first call loads liblcs.so and fails
loudly if it is missing or if no CUDA device is present.  Names follow the C-ABI: lcs_field_create,
lcs_locate, lcs_advect, lcs_cg_ftle, lcs_ftle_host.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblcs.so")

LCS_OK = 0
STATUS_NAMES = {0: "LCS_OK", 1: "LCS_ERR_INVALID_ARG", 2: "LCS_ERR_TIME_RANGE", 3: "LCS_ERR_MESH",
                4: "LCS_ERR_OOM", 5: "LCS_ERR_CUDA", 6: "LCS_ERR_NOT_READY"}
LCS_F32, LCS_F64 = 0, 1
LCS_MESH_CARTESIAN, LCS_MESH_SIMPLEX = 0, 1

EXPORTS = ["lcs_field_create", "lcs_field_set_snapshot", "lcs_field_sync", "lcs_field_destroy", "lcs_field_reserve",
           "lcs_field_set_option", "lcs_field_get_info", "lcs_locate", "lcs_advect", "lcs_advect_series", "lcs_advect_series_reserve", "lcs_advect_early_cg", "lcs_cg_ftle", "lcs_cg_ftle_aux", "lcs_cg_eigen", "lcs_smooth_gaussian", "lcs_smooth_gaussian_static", "lcs_ridge",
           "lcs_ftle_host", "lcs_ftle_series_host", "lcs_measure_peak", "lcs_kernel_launch_count", "lcs_last_error"]
PEAK_KINDS = {"fp32_fma_tflops": 0, "fp64_fma_tflops": 1, "launch_us": 2, "hbm_copy_gbs": 3, "l2_seq_gbs": 4, "l2_sector_gbs": 5,
              "hbm_sector_gbs": 6, "l1_gather_line_gbs": 7, "l1_gather_same_gbs": 8, "l1_gather_spread_gbs": 9,
              "smem_contiguous_gbs": 10, "smem_records_gbs": 11, "smem_records_swizzled_gbs": 12, "smem_records_same_gbs": 13,
              "l1_gather_warp_same_gbs": 14, "l1_gather_warp_line_gbs": 15, "l1_gather_warp_2lines_gbs": 16}


class LcsError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), msg))
        self.status = status


class lcs_field_desc(C.Structure):
    _fields_ = [("dim", C.c_int32), ("kind", C.c_int32),
                ("n", C.c_int32 * 3), ("periodic", C.c_int32 * 3),
                ("origin", C.c_double * 3), ("spacing", C.c_double * 3),
                ("n_vertices", C.c_int64), ("n_cells", C.c_int64),
                ("vertices", C.c_void_p), ("cells", C.c_void_p),
                ("n_snapshots", C.c_int32), ("vel_dtype", C.c_int32),
                ("times", C.c_void_p),
                ("compute_dtype", C.c_int32), ("max_resident_snapshots", C.c_int32)]


_lib = None


def lib():
    """Loads liblcs.so (built in-tree by paper_2209_13775_b200.build).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("liblcs.so not built: run `python -m paper_2209_13775_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.lcs_last_error.restype = C.c_char_p
        L.lcs_kernel_launch_count.restype = C.c_int64
        L.lcs_field_create.argtypes = [C.POINTER(lcs_field_desc), C.POINTER(C.c_void_p)]
        L.lcs_field_set_snapshot.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32]
        L.lcs_field_sync.argtypes = [C.c_void_p]
        L.lcs_field_destroy.argtypes = [C.c_void_p]
        L.lcs_field_destroy.restype = None
        L.lcs_field_reserve.argtypes = [C.c_void_p, C.c_int64, C.c_int64]
        L.lcs_measure_peak.argtypes = [C.c_int32, C.POINTER(C.c_double)]
        L.lcs_field_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
        L.lcs_field_get_info.argtypes = [C.c_void_p, C.c_char_p, C.POINTER(C.c_int64)]
        L.lcs_locate.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_advect.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_double, C.c_double, C.c_double,
                                 C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_advect_series.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int32, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_void_p]
        L.lcs_advect_series_reserve.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_double, C.c_double]
        L.lcs_ftle_series_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_double,
                                           C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_cg_ftle.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_advect_early_cg.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                          C.c_double, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                          C.c_void_p, C.c_void_p]
        L.lcs_cg_ftle_aux.argtypes = [C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                      C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_smooth_gaussian.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                                          C.c_void_p]
        L.lcs_smooth_gaussian_static.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_ridge.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_cg_eigen.argtypes = [C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lcs_ftle_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _check(status):
    if status != LCS_OK:
        raise LcsError(status, lib().lcs_last_error().decode())


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dt(np_dtype):
    return LCS_F64 if np.dtype(np_dtype) == np.float64 else LCS_F32


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _tptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _arr3(vals, ctype, fill, dim=3):
    vals = list(vals) + [fill] * (3 - len(vals))
    return (ctype * 3)(*vals[:3])


def kernel_launch_count() -> int:
    return int(lib().lcs_kernel_launch_count())


def measure_peak(kind) -> float:
    """lcs_measure_peak: kind is an lcs_peak_kind value or a PEAK_KINDS name (TFLOP/s, microseconds or GB/s, see lcs.h)."""
    v = C.c_double()
    _check(lib().lcs_measure_peak(int(PEAK_KINDS.get(kind, kind)), C.byref(v)))
    return float(v.value)


def _n_steps(t0, tf, h) -> int:
    return max(1, int(round((float(tf) - float(t0)) / float(h)))) if h else 1


class Field:
    """lcs_field: mesh + velocity snapshots resident on the device."""

    def __init__(self, dim, kind, times, vel_dtype, compute_dtype, n=(1, 1, 1), origin=(0, 0, 0), spacing=(1, 1, 1),
                 periodic=(0, 0, 0), vertices=None, cells=None, max_resident_snapshots=0):
        self._h = C.c_void_p()
        self.dim, self.kind = int(dim), int(kind)
        self.vel_dtype, self.compute_dtype = np.dtype(vel_dtype), np.dtype(compute_dtype)
        self.times = np.ascontiguousarray(times, dtype=np.float64)
        d = lcs_field_desc()
        d.dim, d.kind = self.dim, self.kind
        for a in range(3):
            d.n[a] = int(n[a]) if a < len(n) else 1
            d.periodic[a] = int(periodic[a]) if a < len(periodic) else 0
            d.origin[a] = float(origin[a]) if a < len(origin) else 0.0
            d.spacing[a] = float(spacing[a]) if a < len(spacing) else 1.0
        self._keep = []
        if self.kind == LCS_MESH_SIMPLEX:
            v = np.ascontiguousarray(vertices, dtype=np.float64)
            c = np.ascontiguousarray(cells, dtype=np.int32)
            d.n_vertices, d.n_cells = v.shape[0], c.shape[0]
            d.vertices, d.cells = _np_ptr(v), _np_ptr(c)
            self.n_nodes = v.shape[0]
        else:
            self.n_nodes = int(d.n[0]) * int(d.n[1]) * int(d.n[2])
        d.n_snapshots = len(self.times)
        d.vel_dtype, d.compute_dtype = _dt(self.vel_dtype), _dt(self.compute_dtype)
        d.times = _np_ptr(self.times)
        d.max_resident_snapshots = int(max_resident_snapshots)
        _check(lib().lcs_field_create(C.byref(d), C.byref(self._h)))

    @classmethod
    def from_workload(cls, w, max_resident_snapshots=0, pinned=False, upload=True):
        """Creates the field of a paper_2209_13775_b200.inputs.Workload and uploads every snapshot."""
        f = cls(w.dim, w.kind, w.times, w.vel.dtype, w.compute_dtype, n=w.n, origin=w.origin, spacing=w.spacing,
                periodic=w.periodic, vertices=w.vertices, cells=w.cells, max_resident_snapshots=max_resident_snapshots)
        if upload:
            vel = w.vel
            if pinned or max_resident_snapshots:
                import torch
                vel_t = torch.from_numpy(np.ascontiguousarray(w.vel)).pin_memory()
                f._keep.append(vel_t)
                vel = vel_t.numpy()
            for s in range(len(w.times)):
                f.set_snapshot(s, vel[s])
            f.sync()
        return f

    def set_snapshot(self, s, vel):
        """vel: numpy array (host) or torch CUDA tensor, [n_nodes][dim] of vel_dtype."""
        if isinstance(vel, np.ndarray):
            assert vel.dtype == self.vel_dtype and vel.flags.c_contiguous and vel.size == self.n_nodes * self.dim
            self._keep.append(vel)
            _check(lib().lcs_field_set_snapshot(self._h, int(s), _np_ptr(vel), 0))
        else:
            assert vel.is_cuda and vel.is_contiguous() and vel.numel() == self.n_nodes * self.dim
            _check(lib().lcs_field_set_snapshot(self._h, int(s), _tptr(vel), 1))

    def sync(self):
        _check(lib().lcs_field_sync(self._h))

    def set_option(self, key, value):
        _check(lib().lcs_field_set_option(self._h, key.encode(), int(value)))

    def reserve(self, n_seeds, n_steps):
        """lcs_field_reserve: set-up call that allocates what lcs_advect needs for up to n_seeds tracers and n_steps steps under
        the current options (the hot calls never allocate).  advect() below calls it, so Python users need not."""
        _check(lib().lcs_field_reserve(self._h, int(n_seeds), int(n_steps)))

    def info(self, key) -> int:
        v = C.c_int64()
        _check(lib().lcs_field_get_info(self._h, key.encode(), C.byref(v)))
        return int(v.value)

    def close(self):
        if self._h:
            lib().lcs_field_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- hot calls (device tensors) ------------------------------------------------------------
    def locate(self, pos, want_bary=False, stream=None):
        """pos: torch CUDA fp64 [n][dim].  Returns cell (int32 [n]) and optionally the weights."""
        import torch
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous()
        n = pos.shape[0]
        cell = torch.empty(n, dtype=torch.int32, device=pos.device)
        nb = self.dim if self.kind == LCS_MESH_CARTESIAN else self.dim + 1
        bary = torch.empty((n, nb), dtype=torch.float64, device=pos.device) if want_bary else None
        _check(lib().lcs_locate(self._h, n, _tptr(pos), _tptr(cell), _tptr(bary), _stream_ptr(stream)))
        return (cell, bary) if want_bary else cell

    def advect(self, seeds, t0, tf, h, flowmap=None, exit_flag=None, exit_step=None, stream=None, want_flags=True, reserve=True):
        """seeds: torch CUDA [n][dim] of compute_dtype.  Returns (flowmap, exit_flag, exit_step).  reserve=False skips the
        lcs_field_reserve call (lcs_advect then fails with LCS_ERR_OOM unless an earlier reservation covers it)."""
        import torch
        tdt = torch.float64 if self.compute_dtype == np.float64 else torch.float32
        assert seeds.is_cuda and seeds.dtype == tdt and seeds.is_contiguous()
        n = seeds.shape[0]
        if flowmap is None:
            flowmap = torch.empty_like(seeds)
        if want_flags:
            if exit_flag is None:
                exit_flag = torch.empty(n, dtype=torch.uint8, device=seeds.device)
            if exit_step is None:
                exit_step = torch.empty(n, dtype=torch.int32, device=seeds.device)
        if reserve and n > 0 and 0 < _n_steps(t0, tf, h) < (1 << 24):
            self.reserve(n, _n_steps(t0, tf, h))             # no-op once the reservation covers the call
        _check(lib().lcs_advect(self._h, n, _tptr(seeds), float(t0), float(tf), float(h), _tptr(flowmap),
                                _tptr(exit_flag), _tptr(exit_step), _stream_ptr(stream)))
        return flowmap, exit_flag, exit_step

    def advect_series(self, seeds, t_start, T, h, flowmaps=None, exit_flags=None, exit_steps=None, stream=None, reserve=True):
        """lcs_advect_series: the same seeds released at every t_start[k], each integrated over T with step h.  Returns
        (flowmaps [n_vol][n][dim], exit_flags [n_vol][n], exit_steps [n_vol][n]) as torch CUDA tensors."""
        import torch
        assert seeds.is_cuda and seeds.is_contiguous()
        n, dim = seeds.shape
        ts = np.ascontiguousarray(t_start, dtype=np.float64)
        nv = int(ts.shape[0])
        if flowmaps is None:
            flowmaps = torch.empty((nv, n, dim), dtype=seeds.dtype, device=seeds.device)
        if exit_flags is None:
            exit_flags = torch.empty((nv, n), dtype=torch.uint8, device=seeds.device)
        if exit_steps is None:
            exit_steps = torch.empty((nv, n), dtype=torch.int32, device=seeds.device)
        if reserve:
            _check(lib().lcs_advect_series_reserve(self._h, n, nv, _np_ptr(ts), float(T), float(h)))
        _check(lib().lcs_advect_series(self._h, n, _tptr(seeds), nv, _np_ptr(ts), float(T), float(h), _tptr(flowmaps), _tptr(exit_flags),
                                       _tptr(exit_steps), _stream_ptr(stream)))
        return flowmaps, exit_flags, exit_steps

    def ftle_host(self, ng, seed_spacing, seed_periodic, period, seeds, t0, tf, h, flowmap=None, exit_flag=None, ftle=None,
                  exit_step=None, cg=None):
        """End-to-end with HOST numpy buffers (H2D + advect + cg_ftle + D2H inside the call); flowmap, exit_flag, exit_step
        and cg are optional outputs."""
        seeds = np.ascontiguousarray(seeds, dtype=self.compute_dtype)
        n = seeds.shape[0]
        if ftle is None:
            ftle = np.empty(n, dtype=self.compute_dtype)
        _check(lib().lcs_ftle_host(self._h, _arr3(ng, C.c_int32, 1), _arr3(seed_spacing, C.c_double, 1.0),
                                   _arr3(seed_periodic, C.c_int32, 0), _arr3(period, C.c_double, 0.0),
                                   _np_ptr(seeds), float(t0), float(tf), float(h), _np_ptr(flowmap), _np_ptr(exit_flag),
                                   _np_ptr(exit_step), _np_ptr(cg), _np_ptr(ftle)))
        return ftle

    def ftle_series_host(self, ng, seed_spacing, seed_periodic, period, seeds, t_start, T, h, ftle=None, cg=None, flowmaps=None,
                         exit_flags=None, exit_steps=None):
        """lcs_ftle_series_host with HOST numpy buffers; returns ftle [n_vol][n]."""
        seeds = np.ascontiguousarray(seeds, dtype=self.compute_dtype)
        ts = np.ascontiguousarray(t_start, dtype=np.float64)
        n, nv = seeds.shape[0], int(ts.shape[0])
        if ftle is None:
            ftle = np.empty((nv, n), dtype=self.compute_dtype)
        _check(lib().lcs_ftle_series_host(self._h, _arr3(ng, C.c_int32, 1), _arr3(seed_spacing, C.c_double, 1.0), _arr3(seed_periodic, C.c_int32, 0),
                                          _arr3(period, C.c_double, 0.0), _np_ptr(seeds), nv, _np_ptr(ts), float(T), float(h), _np_ptr(flowmaps),
                                          _np_ptr(exit_flags), _np_ptr(exit_steps), _np_ptr(cg), _np_ptr(ftle)))
        return ftle


def cg_ftle(dim, ng, seed_spacing, seed_periodic, period, flowmap, exit_flag, T, want_cg=True, want_status=True, stream=None):
    """flowmap: torch CUDA [n][dim] fp32/fp64.  Returns (cg or None, ftle, status or None)."""
    import torch
    assert flowmap.is_cuda and flowmap.is_contiguous()
    n = flowmap.shape[0]
    dtype = LCS_F64 if flowmap.dtype == torch.float64 else LCS_F32
    cg = torch.empty((n, 3 if dim == 2 else 6), dtype=flowmap.dtype, device=flowmap.device) if want_cg else None
    ftle = torch.empty(n, dtype=flowmap.dtype, device=flowmap.device)
    status = torch.empty(n, dtype=torch.uint8, device=flowmap.device) if want_status else None
    _check(lib().lcs_cg_ftle(int(dim), dtype, _arr3(ng, C.c_int32, 1), _arr3(seed_spacing, C.c_double, 1.0),
                             _arr3(seed_periodic, C.c_int32, 0), _arr3(period, C.c_double, 0.0),
                             _tptr(flowmap), _tptr(exit_flag), float(T), _tptr(cg), _tptr(ftle), _tptr(status),
                             _stream_ptr(stream)))
    return cg, ftle, status


def cg_eigen(dim, cg, stream=None):
    """cg: torch CUDA [n][3|6] as returned by cg_ftle.  Returns (evals [n][dim] ascending, evecs [n][dim][dim], row i = unit
    eigenvector of evals[i])."""
    import torch
    assert cg.is_cuda and cg.is_contiguous() and cg.shape[1] == (3 if dim == 2 else 6)
    n = cg.shape[0]
    dtype = LCS_F64 if cg.dtype == torch.float64 else LCS_F32
    evals = torch.empty((n, dim), dtype=cg.dtype, device=cg.device)
    evecs = torch.empty((n, dim, dim), dtype=cg.dtype, device=cg.device)
    _check(lib().lcs_cg_eigen(int(dim), dtype, n, _tptr(cg), _tptr(evals), _tptr(evecs), _stream_ptr(stream)))
    return evals, evecs


def cg_ftle_aux(dim, aux_delta, flow_aux, flag_aux, T, want_cg=True, want_status=True, stream=None):
    """flow_aux: torch CUDA [n][2 dim][dim] (final positions of the auxiliary tracers, see lcs.h); flag_aux [n][2 dim] u8 or
    None.  Returns (cg or None, ftle, status or None)."""
    import torch
    assert flow_aux.is_cuda and flow_aux.is_contiguous()
    n = flow_aux.numel() // (2 * dim * dim)
    dtype = LCS_F64 if flow_aux.dtype == torch.float64 else LCS_F32
    cg = torch.empty((n, 3 if dim == 2 else 6), dtype=flow_aux.dtype, device=flow_aux.device) if want_cg else None
    ftle = torch.empty(n, dtype=flow_aux.dtype, device=flow_aux.device)
    status = torch.empty(n, dtype=torch.uint8, device=flow_aux.device) if want_status else None
    _check(lib().lcs_cg_ftle_aux(int(dim), dtype, n, _arr3(aux_delta, C.c_double, 1.0), _tptr(flow_aux), _tptr(flag_aux), float(T),
                                 _tptr(cg), _tptr(ftle), _tptr(status), _stream_ptr(stream)))
    return cg, ftle, status


def advect_early_cg(field, ng, seed_spacing, seed_periodic, period, seeds, t0, tf, h, every, stream=None):
    """lcs_advect_early_cg: returns (flowmap, exit_flag, exit_step, cg, ftle, t_eff, status), torch CUDA tensors."""
    import torch
    assert seeds.is_cuda and seeds.is_contiguous()
    n, dim = seeds.shape
    F = torch.empty_like(seeds)
    flag = torch.empty(n, dtype=torch.uint8, device=seeds.device)
    es = torch.empty(n, dtype=torch.int32, device=seeds.device)
    cg = torch.empty((n, 3 if dim == 2 else 6), dtype=seeds.dtype, device=seeds.device)
    ftle = torch.empty(n, dtype=seeds.dtype, device=seeds.device)
    t_eff = torch.empty(n, dtype=seeds.dtype, device=seeds.device)
    status = torch.empty(n, dtype=torch.uint8, device=seeds.device)
    if n > 0 and 0 < _n_steps(t0, tf, h) < (1 << 24):
        field.reserve(n, _n_steps(t0, tf, h))
    _check(lib().lcs_advect_early_cg(field._h, _arr3(ng, C.c_int32, 1), _arr3(seed_spacing, C.c_double, 1.0), _arr3(seed_periodic, C.c_int32, 0),
                                     _arr3(period, C.c_double, 0.0), _tptr(seeds), float(t0), float(tf), float(h), int(every), _tptr(F),
                                     _tptr(flag), _tptr(es), _tptr(cg), _tptr(ftle), _tptr(t_eff), _tptr(status), _stream_ptr(stream)))
    return F, flag, es, cg, ftle, t_eff, status


def smooth_gaussian(dim, ng, seed_periodic, sigma, field, stream=None):
    """lcs_smooth_gaussian on a torch CUDA tensor [n]; returns the smoothed field."""
    import torch
    assert field.is_cuda and field.is_contiguous()
    dtype = LCS_F64 if field.dtype == torch.float64 else LCS_F32
    out, work = torch.empty_like(field), torch.empty_like(field)
    _check(lib().lcs_smooth_gaussian(int(dim), dtype, _arr3(ng, C.c_int32, 1), _arr3(seed_periodic, C.c_int32, 0), float(sigma),
                                     _tptr(field), _tptr(out), _tptr(work), _stream_ptr(stream)))
    return out


SMOOTH_STATIC_MAX_BYTES = 16 << 20


def smooth_gaussian_static(dim, ng, seed_periodic, sigma, field, out, stream=None):
    """lcs_smooth_gaussian_static: smoothing with the library's static scratch (no allocation inside the call; the caller supplies
    `out`).  field, out: torch CUDA tensors [n] of the same dtype, distinct.  Returns out."""
    import torch
    assert field.is_cuda and field.is_contiguous() and out.is_cuda and out.is_contiguous() and out.dtype == field.dtype
    dtype = LCS_F64 if field.dtype == torch.float64 else LCS_F32
    _check(lib().lcs_smooth_gaussian_static(int(dim), dtype, _arr3(ng, C.c_int32, 1), _arr3(seed_periodic, C.c_int32, 0), float(sigma),
                                            _tptr(field), _tptr(out), _stream_ptr(stream)))
    return out


def ridge(dim, ng, seed_spacing, seed_periodic, kappa_min, s_min, field, stream=None):
    """lcs_ridge on a torch CUDA tensor [n]; returns (kappa, d, mask)."""
    import torch
    assert field.is_cuda and field.is_contiguous()
    dtype = LCS_F64 if field.dtype == torch.float64 else LCS_F32
    kappa, d = torch.empty_like(field), torch.empty_like(field)
    mask = torch.empty(field.numel(), dtype=torch.uint8, device=field.device)
    _check(lib().lcs_ridge(int(dim), dtype, _arr3(ng, C.c_int32, 1), _arr3(seed_spacing, C.c_double, 1.0), _arr3(seed_periodic, C.c_int32, 0),
                           float(kappa_min), float(s_min), _tptr(field), _tptr(kappa), _tptr(d), _tptr(mask), _stream_ptr(stream)))
    return kappa, d, mask
