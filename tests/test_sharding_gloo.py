"""Multi-process (world_size 2, gloo, CPU) test of the N > 1 path's host logic: event sharding + the one
histogram all-reduce.  The per-rank partial histogram is filled here by the
test oracle (the CUDA kernels need a GPU; their parity is tests/test_parity_gpu.py); what is under test is
``paper_1311_7579_b200.sharding``: the slices partition the sample and the reduced histogram equals the
single-process one to summation-order rounding."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

from paper_1311_7579_b200 import sharding
from paper_1311_7579_b200 import workloads as wl

torch = pytest.importorskip("torch")


@pytest.mark.parametrize("n,world,align", [(0, 1, 2), (1, 2, 2), (2, 2, 2), (7, 3, 2), (1000, 8, 2), (1001, 8, 2),
                                           (10_000_000, 8, 2), (13, 4, 1), (5, 8, 2)])
def test_shard_bounds_partition(n, world, align):
    prev = 0
    sizes = []
    for r in range(world):
        b, e = sharding.shard_bounds(n, r, world, align)
        assert b == prev and b <= e <= n
        assert b % align == 0 or b == n
        sizes.append(e - b)
        prev = e
    assert prev == n
    assert max(sizes) - min(sizes) <= 2 * align - 1


def test_shard_bounds_rejects():
    with pytest.raises(ValueError):
        sharding.shard_bounds(10, 2, 2)
    with pytest.raises(ValueError):
        sharding.shard_bounds(-1, 0, 1)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n: int, out_dir: str):
    import torch.distributed as dist

    import oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        par = oracle.Params(**wl.table1())
        et, er, w0, ch = wl.events(n, seed=2)        # every rank regenerates the same seeded sample
        edges = wl.bin_edges()

        def fill(a, b, c, d, s, e, hist_out=None):   # stands in for osc_reweight_bin on this rank's device
            return torch.from_numpy(oracle.reweight_bin(par, a, b, c, d, s, e))

        h = sharding.sharded_reweight_bin(et, er, w0, ch, 1.03, edges, rank, world, fill)
        np.save(os.path.join(out_dir, f"hist_{rank}.npy"), h.numpy())
    finally:
        dist.destroy_process_group()


def test_world2_histogram_allreduce(tmp_path):
    import torch.multiprocessing as mp

    import oracle

    n, world = 20_001, 2
    mp.spawn(_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    par = oracle.Params(**wl.table1())
    et, er, w0, ch = wl.events(n, seed=2)
    ref = oracle.reweight_bin(par, et, er, w0, ch, 1.03, wl.bin_edges())
    h0 = np.load(tmp_path / "hist_0.npy")
    h1 = np.load(tmp_path / "hist_1.npy")
    assert np.array_equal(h0, h1)                    # all-reduce leaves the same sum on every rank
    assert np.array_equal(h0 == 0.0, ref == 0.0)
    nz = ref != 0.0
    assert np.max(np.abs(h0[nz] - ref[nz]) / ref[nz]) <= 1e-13


def _scan_worker(rank: int, world: int, port: int, n: int, out_dir: str):
    import torch.distributed as dist

    import oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        pts = wl.scan_points()[:80]                  # 2.5 groups of 32: the ranks own 64 and 16 points
        et, er, w0, ch = wl.events(n, seed=3)
        edges = wl.bin_edges()

        def batch(p, a, b, c, d, s, e):              # stands in for osc_reweight_bin_batch on this rank's device
            if len(p) == 0:
                return torch.empty((0, 4, edges.size - 1), dtype=torch.float64)
            return torch.from_numpy(oracle.reweight_bin_batch([oracle.Params(**q) for q in p], a, b, c, d, s, e))

        h = sharding.sharded_scan(pts, et, er, w0, ch, 1.0, edges, rank, world, batch)
        np.save(os.path.join(out_dir, f"scan_{rank}.npy"), h.numpy())
    finally:
        dist.destroy_process_group()


def test_world2_scan_sharded_by_points(tmp_path):
    import torch.multiprocessing as mp

    import oracle

    n, world = 501, 2
    mp.spawn(_scan_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    pts = wl.scan_points()[:80]
    et, er, w0, ch = wl.events(n, seed=3)
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, wl.bin_edges())
    h0 = np.load(tmp_path / "scan_0.npy")
    h1 = np.load(tmp_path / "scan_1.npy")
    assert h0.shape == (80, 4, 50)
    assert np.array_equal(h0, h1) and np.array_equal(h0, ref)    # no arithmetic across ranks: bit-identical
    assert sharding.shard_bounds(80, 0, 2, align=32) == (0, 64) and sharding.shard_bounds(80, 1, 2, align=32) == (64, 80)
