"""lcs_smooth_gaussian_static: the entry point that allocates nothing (scratch in a file-scope device array of the library,
16 MiB), for callers that cannot call cudaMalloc.  Collected last on purpose (the file name sorts after every other test file):
it shares a process-wide static array, and a failure here must not hide other tests under `pytest -x`.

Checks, on two calls in a row that reuse the (dirty) scratch: 2D fp64 non-periodic with undefined (NaN) seeds, then 3D fp32 periodic
of a different size: the output equals lcs_smooth_gaussian's (the existing path, itself checked against oracle rule O11 in
test_gpu_parity.py) within that test's tolerances, and the oracle's; the device's free memory does not change across the calls;
sizes beyond the static maximum are rejected with LCS_ERR_INVALID_ARG."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lcs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2209_13775_b200 import build, lcs as L
    build.build()
    L.lib()
    return L


def _field(ng, dtype, seed, nan_every=0):
    """A smooth scalar field on the seed grid plus noise (synthetic FTLE stand-in), optionally with undefined seeds."""
    rng = np.random.default_rng(seed)
    axes = np.meshgrid(*[np.linspace(0.0, 1.0, m, endpoint=False) for m in ng[::-1]], indexing="ij")
    f = sum(np.sin(2.0 * np.pi * (k + 1) * a + 0.3 * k) for k, a in enumerate(axes)) + 0.1 * rng.standard_normal(axes[0].shape)
    f = f.reshape(-1).astype(dtype)
    if nan_every:
        f[::nan_every] = np.nan
    return f


def test_static_scratch_smoothing_matches_the_existing_path_twice(lcs, oracle):
    import torch
    cases = [(2, (211, 97, 1), (0, 0, 0), np.float64, 1.7, 53, 1e-13),          # first call: 2D fp64, open, NaN seeds
             (3, (61, 45, 38), (1, 1, 1), np.float32, 0.9, 0, 2e-6),            # second call: 3D fp32 periodic, another size, dirty scratch
             (2, (211, 97, 1), (0, 0, 0), np.float64, 1.7, 53, 1e-13)]          # and the first one again
    fields = [torch.from_numpy(_field(ng[:dim], dt, 100 + k, nan)).cuda() for k, (dim, ng, per, dt, sigma, nan, tol) in enumerate(cases)]
    outs = [torch.full_like(f, -7.0) for f in fields]
    refs = [lcs.smooth_gaussian(dim, ng, per, sigma, f) for (dim, ng, per, dt, sigma, nan, tol), f in zip(cases, fields)]   # existing path
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (dim, ng, per, dt, sigma, nan, tol), f, o in zip(cases, fields, outs):
        lcs.smooth_gaussian_static(dim, ng, per, sigma, f, o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                                 # nothing was allocated or freed inside the calls
    for (dim, ng, per, dt, sigma, nan, tol), f, o, r in zip(cases, fields, outs, refs):
        got, ref = o.cpu().numpy().astype(np.float64), r.cpu().numpy().astype(np.float64)
        assert np.array_equal(np.isnan(got), np.isnan(ref))
        ok = np.isfinite(ref)
        assert ok.sum() > 1000 and np.max(np.abs(got[ok] - ref[ok])) <= tol * max(1.0, np.abs(ref[ok]).max())
        orc = oracle.smooth_gaussian(dim, ng[:dim], per[:dim], sigma, f.cpu().numpy().astype(np.float64))
        assert np.array_equal(np.isnan(got), np.isnan(orc)) and np.max(np.abs(got[ok] - orc[ok])) <= tol * max(1.0, np.abs(orc[ok]).max())
    assert np.isnan(outs[0].cpu().numpy()).sum() > 10


def test_static_scratch_limits_and_arguments(lcs):
    import torch
    lim32 = lcs.SMOOTH_STATIC_MAX_BYTES // 4
    # exactly at the limit (fp32): accepted
    f = torch.zeros(lim32, dtype=torch.float32, device="cuda")
    o = torch.empty_like(f)
    lcs.smooth_gaussian_static(3, (256, 128, 128), (0, 0, 0), 1.0, f, o)
    torch.cuda.synchronize()
    assert float(o.abs().max()) == 0.0
    # one row beyond it, and the same seed count in fp64: rejected, with the limit in the message
    f2 = torch.zeros(256 * 128 * 129, dtype=torch.float32, device="cuda")
    with pytest.raises(lcs.LcsError) as e:
        lcs.smooth_gaussian_static(3, (256, 128, 129), (0, 0, 0), 1.0, f2, torch.empty_like(f2))
    assert e.value.status == 1 and "static scratch" in str(e.value)
    f3 = torch.zeros(lim32, dtype=torch.float64, device="cuda")
    with pytest.raises(lcs.LcsError) as e:
        lcs.smooth_gaussian_static(3, (256, 128, 128), (0, 0, 0), 1.0, f3, torch.empty_like(f3))
    assert e.value.status == 1
    g = torch.zeros(64, dtype=torch.float32, device="cuda")
    for bad in (dict(sigma=0.0), dict(sigma=30.0)):
        with pytest.raises(lcs.LcsError):
            lcs.smooth_gaussian_static(2, (8, 8, 1), (0, 0, 0), bad["sigma"], g, torch.empty_like(g))
    with pytest.raises(lcs.LcsError):
        lcs.smooth_gaussian_static(2, (8, 8, 1), (0, 0, 0), 1.0, g, g)            # field and out must differ
