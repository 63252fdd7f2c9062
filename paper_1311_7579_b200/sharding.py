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


def sharded_scan(points, E_true, E_reco, w0, channel, energy_scale, bin_edges, rank: int, world: int, batch_fn,
                 group=None):
    """Parameter scan sharded by POINTS ("for scans, sharding parameter points instead needs no
    collective (gather only)"): every rank holds all events, runs ``batch_fn`` (``osc_reweight_bin_batch`` of the
    binding on GPUs) on its contiguous slice of the point list, and the slices are concatenated with one all-gather.

    Slices are cut with ``align=32`` so that the groups of a scan grid (points that differ only in theta23 / delta_cp,
    32 per dm2_32 value in configs[3]) stay whole on one rank and the factorised kernel keeps its full lanes.
    Returns the [n_points, 4, n_bins] tensor on every rank.
    """
    import torch
    import torch.distributed as dist

    n_points = len(points)
    b, e = shard_bounds(n_points, rank, world, align=32)
    part = batch_fn(points[b:e], E_true, E_reco, w0, channel, energy_scale, bin_edges)
    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1):
        return part
    # ranks may own different numbers of points and all_gather wants equal shapes: pad to the largest slice
    sizes = [hi - lo for lo, hi in (shard_bounds(n_points, r, world, align=32) for r in range(world))]
    tail = tuple(part.shape[1:])
    padded = torch.zeros((max(sizes),) + tail, dtype=part.dtype, device=part.device)
    padded[:e - b] = part
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    return torch.cat([q[:m] for q, m in zip(parts, sizes)], dim=0)
