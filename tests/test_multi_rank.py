"""N > 1 path of bench.py on CPU (gloo, world_size 2): the path shards with no data-path collective -- every rank
integrates its own FTLE volume -- so what ranks share is only the reduction of the timing
(MAX over ranks) and of the work (SUM).  The kernels themselves need a GPU and are covered by the -m gpu tests."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms, steps, seeds = bench.reduce_over_ranks(100.0 + 25.0 * rank, 1000.0 * (rank + 1), 64.0, "cpu", world)
        out.put((rank, ms, steps, seeds))
    finally:
        dist.destroy_process_group()


def test_reduce_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, steps, seeds in res:
        assert ms == 125.0 and steps == 3000.0 and seeds == 128.0      # max time, summed work, on every rank


def test_reduce_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(12.5, 7.0, 3.0, "cpu", 1) == (12.5, 7.0, 3.0)


def test_rank_shards_are_independent_volumes_of_equal_size(monkeypatch):
    """Weak scaling: bench.make_workload(3, rank) gives rank r the seed grid released at its own t0 over the same T.  The eight
    windows of one node are distinct, lie inside the snapshot times, have the same number of steps (same work per rank) and
    share the seeds and the field (replicated, no data-path collective)."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2209_13775_b200 import inputs as I
    small = I.config3(ngrid=8, nn=8)
    monkeypatch.setattr(I, "config3", lambda *a, **k: small)
    seen = []
    for rank in range(8):
        w, runs = bench.make_workload(3, rank)
        assert w is small and len(runs) == 1
        t0, tf, h = runs[0]
        assert w.times[0] <= t0 < tf <= w.times[-1] + 1e-12 and h == w.h
        assert int(round((tf - t0) / h)) == w.n_steps
        seen.append((t0, tf))
    assert len(set(seen)) == 8
    # the single-volume configs give every rank the same, complete workload (replicas: they do not shard further)
    for cfg, name in ((1, "config1"), (2, "config2")):
        tiny = getattr(I, name)(ng=(8, 4)) if cfg == 1 else I.config2(ng=(8, 4), lattice=(9, 5))
        monkeypatch.setattr(I, name, lambda *a, _t=tiny, **k: _t)
        assert bench.make_workload(cfg, 0)[1] == bench.make_workload(cfg, 5)[1]


# -------------------------------------------------------------------------------------------------
# one volume across ranks: seed slabs + one halo layer of the flow map (paper_2209_13775_b200/shard.py)
def test_slab_ranges_and_neighbours():
    sys.path.insert(0, ROOT)
    from paper_2209_13775_b200 import shard
    for n, world in ((256, 8), (10, 3), (7, 7), (5, 2)):
        r = [shard.slab_range(n, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == n and all(r[k][1] == r[k + 1][0] for k in range(world - 1))
        sizes = [b - a for a, b in r]
        assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
    assert shard.neighbours(0, 4, False) == (None, 1) and shard.neighbours(3, 4, False) == (2, None)
    assert shard.neighbours(0, 4, True) == (3, 1) and shard.neighbours(3, 4, True) == (2, 0) and shard.neighbours(0, 1, True) == (0, 0)


def _halo_worker(rank, world, port, periodic, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_2209_13775_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nz, plane, dim, period = 7, 12, 3, 6.5
        g = torch.Generator().manual_seed(7)
        F = torch.rand((nz, plane, dim), generator=g, dtype=torch.float32)          # the global flow map, same on every rank
        flag = (torch.rand((nz, plane), generator=g) < 0.2).to(torch.uint8)
        k0, k1 = shard.slab_range(nz, rank, world)
        lo, hi = shard.exchange_halo(F[k0:k1].contiguous(), flag[k0:k1].contiguous(), rank, world, periodic)
        Fe, fe, n_lo = shard.extend_with_halo(F[k0:k1], flag[k0:k1], lo, hi, dim - 1, period, periodic and rank == 0, periodic and rank == world - 1)
        # what the extended slab must be, cut from the global arrays
        idx = list(range(k0 - 1, k1 + 1))
        keep = [k for k in idx if periodic or 0 <= k < nz]
        ref_F = torch.stack([F[k % nz].clone() for k in keep])
        for j, k in enumerate(keep):
            if k < 0: ref_F[j, :, dim - 1] -= period
            if k >= nz: ref_F[j, :, dim - 1] += period
        ref_f = torch.stack([flag[k % nz] for k in keep])
        ok = bool(torch.equal(Fe, ref_F) and torch.equal(fe, ref_f) and n_lo == (1 if keep[0] == k0 - 1 else 0))
        out.put((rank, ok, tuple(Fe.shape)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, False), (2, True), (3, True)])
def test_halo_exchange_gloo(world, periodic):
    """Every rank's slab, extended by the layers it receives, equals the same layers cut from the global flow map (with the
    period added across the seam): world 2 open, world 2 periodic (both neighbours are the same rank), world 3 periodic."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() + 17 * world + int(periodic)) % 2000
    procs = [ctx.Process(target=_halo_worker, args=(r, world, port, periodic, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in res), res
