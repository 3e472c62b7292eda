"""Helpers shared by the GPU parity tests: run the CUDA path (through the C-ABI binding) and the CPU oracle
on the same seeded workload and apply BASELINE.json's gates."""
import numpy as np


def gpu_run(w, seeds=None, max_resident_snapshots=0, options=None, t0=None, tf=None, h=None, field=None):
    import torch
    from paper_2209_13775_b200 import lcs
    f = field or lcs.Field.from_workload(w, max_resident_snapshots=max_resident_snapshots)
    for k, v in (options or {}).items():
        f.set_option(k, v)
    s = w.seeds() if seeds is None else np.ascontiguousarray(seeds, dtype=w.compute_dtype)
    sd = torch.from_numpy(s).cuda()
    F, flag, es = f.advect(sd, w.t0 if t0 is None else t0, w.tf if tf is None else tf, w.h if h is None else h)
    torch.cuda.synchronize()
    return f, sd, F, flag, es


def gpu_cg(w, F, flag, T=None):
    from paper_2209_13775_b200 import lcs
    return lcs.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, F, flag, (w.tf - w.t0) if T is None else T)


def oracle_run(oracle, w, seeds=None, t0=None, tf=None, h=None):
    f = oracle.OracleField.from_workload(w)
    s = w.seeds() if seeds is None else np.ascontiguousarray(seeds, dtype=w.compute_dtype)
    F, flag, es = f.advect(s.astype(np.float64), w.t0 if t0 is None else t0, w.tf if tf is None else tf, w.h if h is None else h)
    return f, F, flag, es


def oracle_cg(oracle, w, F, flag, T=None):
    return oracle.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, F, flag, (w.tf - w.t0) if T is None else T)


def gate_fp64(Fg, Fo, ftle_g, ftle_o, T, flag_g, flag_o, es_g=None, es_o=None):
    """north_star: non-chaotic fp64 flow maps within 1e-10 absolute, FTLE within 1e-8 relative
    (|d sigma| <= 1e-8 |sigma_ref| + 1e-10/|T| so that sigma ~ 0 is testable; DESIGN reading #24)."""
    assert np.array_equal(flag_g, flag_o)
    if es_g is not None:
        assert np.array_equal(es_g, es_o)
    err = np.max(np.abs(Fg - Fo))
    assert err <= 1e-10, err
    ok = np.isfinite(ftle_o)
    assert np.array_equal(np.isfinite(ftle_g), ok)
    d = np.abs(ftle_g[ok] - ftle_o[ok])
    assert np.all(d <= 1e-8 * np.abs(ftle_o[ok]) + 1e-10 / abs(T)), d.max()
    return err


def gate_statistical(Fg, Fo, ftle_g, ftle_o, L, flag_g, flag_o):
    """north_star: chaotic / fp32 configs: >= 99.9% of seeds with flow-map error <= 1e-3 L (exit-flag
    mismatches count against the 0.1%), median FTLE relative error <= 1e-3 against the fp64 oracle."""
    err = np.linalg.norm(Fg.astype(np.float64) - Fo, axis=1)
    bad = (err > 1e-3 * L) | (flag_g != flag_o)
    frac_ok = 1.0 - bad.mean()
    assert frac_ok >= 0.999, frac_ok
    ok = np.isfinite(ftle_o) & np.isfinite(ftle_g)
    assert ok.sum() >= 0.99 * np.isfinite(ftle_o).sum()
    rel = np.abs(ftle_g[ok].astype(np.float64) - ftle_o[ok]) / np.maximum(np.abs(ftle_o[ok]), 1e-300)
    med = np.median(rel) if ok.any() else 0.0
    assert med <= 1e-3, med
    return dict(frac_ok=float(frac_ok), median_ftle_rel=float(med), mean_err=float(err.mean()), max_err=float(err.max()),
                p999_err=float(np.quantile(err, 0.999)))
