"""One FTLE volume across several GPUs: seed slabs along the slowest grid axis plus one halo layer of the flow map.

Paper: tracers are independent, so the advection of a seed grid splits across devices with no exchange; the
only coupling is the central difference of the flow map, which reaches one seed into the neighbouring slab.  "For
significantly larger ... tracer grids, one will overflow the global memory": this is the split for that case
(DESIGN.md 9).

Rank r owns the seed layers [k0, k1) of the last grid axis.  After lcs_advect of its own seeds it receives the first / last layer
of flow map and exit flags of its neighbours (torch.distributed point-to-point: NCCL over NVLink on GPUs, gloo in the CPU test),
adds the period to the component along the split axis of a layer that arrives across a periodic seam (reading #13:
stored positions are never wrapped), runs lcs_cg_ftle on the extended slab with the split axis declared non-periodic, and keeps
its own layers.  The result equals the single-device computation (bit for bit away from a periodic seam; to the rounding of
`F + period` in the flow map's type for the two layers next to it).

No arithmetic of the method lives here: slab bookkeeping, the exchange and argument marshalling only.
"""
from __future__ import annotations

from typing import Optional, Tuple


def slab_range(n_layers: int, rank: int, world: int) -> Tuple[int, int]:
    """Layers [k0, k1) of rank `rank`: contiguous, balanced to within one layer, every rank non-empty when n_layers >= world."""
    base, rem = divmod(int(n_layers), int(world))
    k0 = rank * base + min(rank, rem)
    return k0, k0 + base + (1 if rank < rem else 0)


def neighbours(rank: int, world: int, periodic: bool) -> Tuple[Optional[int], Optional[int]]:
    """(rank holding the layers below mine, rank holding the layers above mine); None at an open end of the grid."""
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank + 1 < world else (0 if periodic else None)
    return lo, hi


def extend_with_halo(F, flag, lo_layer, hi_layer, axis_comp: int, period: float, lo_wrapped: bool, hi_wrapped: bool):
    """F: [nl][plane][dim], flag: [nl][plane] (torch tensors).  lo_layer / hi_layer: (F [plane][dim], flag [plane]) of the
    neighbouring slabs or None.  A layer that arrived across the periodic seam gets -/+ period on component `axis_comp`.
    Returns (F_ext, flag_ext, n_lo) with n_lo = 1 if a layer was prepended."""
    import torch
    parts_F, parts_f, n_lo = [], [], 0
    if lo_layer is not None:
        Fl = lo_layer[0].clone()
        if lo_wrapped:
            Fl[:, axis_comp] -= period
        parts_F.append(Fl.unsqueeze(0)); parts_f.append(lo_layer[1].unsqueeze(0)); n_lo = 1
    parts_F.append(F); parts_f.append(flag)
    if hi_layer is not None:
        Fh = hi_layer[0].clone()
        if hi_wrapped:
            Fh[:, axis_comp] += period
        parts_F.append(Fh.unsqueeze(0)); parts_f.append(hi_layer[1].unsqueeze(0))
    return torch.cat(parts_F, 0).contiguous(), torch.cat(parts_f, 0).contiguous(), n_lo


def exchange_halo(F, flag, rank: int, world: int, periodic: bool, group=None):
    """Sends my first layer down and my last layer up, receives the matching layers of the neighbours.
    F: [nl][plane][dim], flag: [nl][plane] u8.  Returns (lo_layer, hi_layer), each (F [plane][dim], flag [plane]) or None."""
    import torch
    import torch.distributed as dist
    lo, hi = neighbours(rank, world, periodic)
    if world == 1:
        # a single slab: its own far layers are its periodic neighbours
        return ((F[-1], flag[-1]) if periodic else None), ((F[0], flag[0]) if periodic else None)
    ops, recv = [], {}
    first = (F[0].contiguous(), flag[0].contiguous())
    last = (F[-1].contiguous(), flag[-1].contiguous())
    if lo is not None:
        recv["lo"] = (torch.empty_like(first[0]), torch.empty_like(first[1]))
        ops += [dist.P2POp(dist.isend, first[0], lo, group), dist.P2POp(dist.isend, first[1], lo, group),
                dist.P2POp(dist.irecv, recv["lo"][0], lo, group), dist.P2POp(dist.irecv, recv["lo"][1], lo, group)]
    if hi is not None:
        recv["hi"] = (torch.empty_like(last[0]), torch.empty_like(last[1]))
        ops += [dist.P2POp(dist.isend, last[0], hi, group), dist.P2POp(dist.isend, last[1], hi, group),
                dist.P2POp(dist.irecv, recv["hi"][0], hi, group), dist.P2POp(dist.irecv, recv["hi"][1], hi, group)]
    if world == 2 and periodic and lo == hi:
        # two ranks on a periodic axis: both of my neighbours are the same rank; what I receive "from below" is ITS last layer
        # and "from above" its first.  Tag the four transfers by posting them in a fixed order on both sides: lower rank sends
        # (first, last) and receives (last-of-peer, first-of-peer) in the order the peer sends them.
        peer = lo
        recv = {"lo": (torch.empty_like(first[0]), torch.empty_like(first[1])), "hi": (torch.empty_like(last[0]), torch.empty_like(last[1]))}
        ops = [dist.P2POp(dist.isend, first[0], peer, group), dist.P2POp(dist.isend, first[1], peer, group),
               dist.P2POp(dist.isend, last[0], peer, group), dist.P2POp(dist.isend, last[1], peer, group),
               dist.P2POp(dist.irecv, recv["hi"][0], peer, group), dist.P2POp(dist.irecv, recv["hi"][1], peer, group),
               dist.P2POp(dist.irecv, recv["lo"][0], peer, group), dist.P2POp(dist.irecv, recv["lo"][1], peer, group)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    return recv.get("lo"), recv.get("hi")


def slab_seed_grid(ng, seed_spacing, seed_lo, k0: int, k1: int, dim: int):
    """(ng_slab, lo_slab) of the seed layers [k0, k1) along the last axis of a cell-centred structured seed grid."""
    ng_s = list(ng); lo_s = list(seed_lo)
    ng_s[dim - 1] = k1 - k0
    lo_s[dim - 1] = seed_lo[dim - 1] + k0 * seed_spacing[dim - 1]
    return tuple(ng_s), tuple(lo_s)


def cg_ftle_slab(lcs, dim, ng, seed_spacing, seed_periodic, period, F_slab, flag_slab, T, rank, world, group=None,
                 want_cg=True, want_status=False):
    """F_slab: torch CUDA [n_slab][dim] (seed order of the slab, axis 0 fastest), flag_slab [n_slab] u8: the outputs of
    lcs_advect on this rank's layers of the last grid axis.  Exchanges one halo layer, runs lcs_cg_ftle on the extended slab
    and returns (cg, ftle, status) for the rank's own seeds."""
    ax = dim - 1
    plane = 1
    for a in range(ax):
        plane *= int(ng[a])
    nl = F_slab.shape[0] // plane
    F3 = F_slab.view(nl, plane, dim)
    f3 = flag_slab.view(nl, plane)
    per = bool(seed_periodic[ax])
    lo_layer, hi_layer = exchange_halo(F3, f3, rank, world, per, group)
    lo_r, hi_r = neighbours(rank, world, per)
    lo_wrapped = per and (world == 1 or rank == 0)
    hi_wrapped = per and (world == 1 or rank == world - 1)
    Fe, fe, n_lo = extend_with_halo(F3, f3, lo_layer, hi_layer, ax, float(period[ax]), lo_wrapped, hi_wrapped)
    ng_e = list(ng) + [1] * (3 - len(ng))
    ng_e[ax] = Fe.shape[0]
    per_e = list(seed_periodic) + [0] * (3 - len(seed_periodic))
    per_e[ax] = 0                                         # the halo layers stand in for the neighbours across the slab faces
    cg, ftle, status = lcs.cg_ftle(dim, tuple(ng_e), seed_spacing, tuple(per_e), period, Fe.view(-1, dim), fe.view(-1), T,
                                   want_cg=want_cg, want_status=want_status)
    a, b = n_lo * plane, (n_lo + nl) * plane
    return (cg[a:b] if cg is not None else None), ftle[a:b], (status[a:b] if status is not None else None)
