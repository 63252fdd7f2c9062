"""Multi-GPU plumbing of the path: which events a rank owns and the one
collective the path has.

Events are independent ("the events are independent of each other"), so the path shards by events:
rank r of W owns one contiguous slice, fills a partial histogram with ``osc_reweight_bin`` / ``osc_reweight_bin_batch``
on its own GPU, and the partials are summed with ONE all-reduce of 4 * n_bins doubles (per parameter point).  The
per-event probability arrays of ``osc_prob`` need no collective at all.

Nothing here does arithmetic of the method; ``torch.distributed`` (NCCL on GPUs, gloo in the CPU tests) is plumbing.
"""
from __future__ import annotations

from typing import Tuple


def shard_bounds(n: int, rank: int, world: int, align: int = 2) -> Tuple[int, int]:
    """[begin, end) of rank ``rank``'s contiguous slice of ``n`` events.

    Slices are balanced to within ``2 * align - 1`` events and every begin is a multiple of ``align`` (default 2: keeps the
    16-byte alignment of fp64 arrays that the kernels' 128-bit loads want).  The slices partition [0, n) exactly.
    """
    if world < 1 or not (0 <= rank < world):
        raise ValueError(f"bad rank/world: {rank}/{world}")
    if n < 0 or align < 1:
        raise ValueError("n must be >= 0 and align >= 1")
    units = (n + align - 1) // align            # number of align-sized groups (last may be partial)
    base, extra = divmod(units, world)
    u0 = rank * base + min(rank, extra)
    u1 = u0 + base + (1 if rank < extra else 0)
    return min(u0 * align, n), min(u1 * align, n)


def allreduce_hist(hist, group=None):
    """Sum the ranks' partial histograms in place (one collective; no-op outside a process group).

    ``hist`` is a torch tensor ([4, n_bins] or [n_points, 4, n_bins], fp64) on the device of the backend in use.
    Returns ``hist``.
    """
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(hist, op=dist.ReduceOp.SUM, group=group)
    return hist


def sharded_reweight_bin(E_true, E_reco, w0, channel, energy_scale, bin_edges, rank: int, world: int,
                         reweight_fn, hist_out=None, group=None):
    """Histogram of the full sample from per-rank partials: ``reweight_fn`` (``osc_reweight_bin`` of the binding on
    GPUs) runs on this rank's slice of the event arrays, then ``allreduce_hist`` sums over ranks.

    The event arrays are the FULL arrays (or views of them) resident on this rank; only [begin, end) is touched.
    """
    b, e = shard_bounds(E_true.shape[0], rank, world)
    part = reweight_fn(E_true[b:e], E_reco[b:e], w0[b:e], channel[b:e], energy_scale, bin_edges, hist_out=hist_out)
    return allreduce_hist(part, group)


GROUP_FIELDS = ("sin2_th12", "sin2_th13", "dm2_32", "dm2_21", "rho_g_cm3", "L_km", "hierarchy")


def _field(p, name):
    return p[name] if isinstance(p, dict) else getattr(p, name)


def scan_partition(points, world: int, lanes: int = 32):
    """Which points of a parameter list each rank takes: ``[indices of rank 0, indices of rank 1, ...]``.

    The batched call does the eigen-solve once per GROUP -- the points that agree in everything except sin2_th23 and
    delta_cp (``GROUP_FIELDS``; include/osc.h, osc_reweight_bin_batch) -- and serves 32 points of a group per warp pass.
    So whole groups go to ranks: a group is cut only when there are fewer groups than ranks would need, and then into
    pieces of a multiple of ``lanes`` points.  configs[3] orders its 32 x 32 grid as p = 32 i_th23 + j_dm2, i.e. the 32
    points of a group are strided by 32 in the list: contiguous slices would leave every rank with all 32 groups at
    32 / world points each, repeat every eigen-solve on every rank and run the factorised kernel with mostly empty
    lanes.  Pieces are handed out largest first to the least loaded rank (ties: lowest rank), so the partition is a
    deterministic function of the list; inside a rank the points keep their order of the list."""
    if world < 1:
        raise ValueError("world must be >= 1")
    groups = {}
    for i, p in enumerate(points):
        groups.setdefault(tuple(_field(p, f) for f in GROUP_FIELDS), []).append(i)
    pieces = list(groups.values())
    # fewer pieces than ranks: cut the largest pieces at multiples of `lanes` while that gives another rank work
    while pieces and len(pieces) < world:
        pieces.sort(key=lambda g: (-len(g), g[0]))
        big = pieces[0]
        if len(big) <= lanes:
            break
        half = max(lanes, (len(big) // 2 + lanes - 1) // lanes * lanes)
        pieces = [big[:half], big[half:]] + pieces[1:]
    pieces.sort(key=lambda g: (-len(g), g[0]))
    owned = [[] for _ in range(world)]
    for g in pieces:
        r = min(range(world), key=lambda k: (len(owned[k]), k))
        owned[r].extend(g)
    return [sorted(o) for o in owned]


def sharded_scan(points, E_true, E_reco, w0, channel, energy_scale, bin_edges, rank: int, world: int, batch_fn,
                 group=None):
    """Parameter scan sharded by POINTS ("for scans, sharding parameter points instead needs no
    collective (gather only)"): every rank holds all events, runs ``batch_fn`` (``osc_reweight_bin_batch`` of the
    binding on GPUs) on the points ``scan_partition`` gives it -- whole eigen-problem groups, so no eigen-solve is
    repeated across ranks and the factorised kernel keeps full lanes -- and the slices are put back into the order of the
    list after one all-gather.  No arithmetic crosses ranks.  Returns the [n_points, 4, n_bins] tensor on every rank."""
    import torch
    import torch.distributed as dist

    n_points = len(points)
    owned = scan_partition(points, world)
    mine = owned[rank]
    part = batch_fn([points[i] for i in mine], E_true, E_reco, w0, channel, energy_scale, bin_edges)
    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1):
        out = torch.empty((n_points,) + tuple(part.shape[1:]), dtype=part.dtype, device=part.device)
        out[torch.as_tensor(mine, dtype=torch.long, device=part.device)] = part
        return out
    # ranks may own different numbers of points and all_gather wants equal shapes: pad to the largest slice
    sizes = [len(o) for o in owned]
    tail = tuple(part.shape[1:])
    padded = torch.zeros((max(sizes),) + tail, dtype=part.dtype, device=part.device)
    padded[:len(mine)] = part
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    out = torch.empty((n_points,) + tail, dtype=part.dtype, device=part.device)
    for q, o in zip(parts, owned):
        if o:
            out[torch.as_tensor(o, dtype=torch.long, device=part.device)] = q[:len(o)]
    return out
