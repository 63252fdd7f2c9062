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
        pts = wl.scan_points()[:80]                  # 32 dm2_32 groups of 2 or 3 points each, strided through the list
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


@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_scan_partition_keeps_groups_whole(world):
    """configs[3] (p = 32 i_th23 + j_dm2: the 32 points of a dm2_32 group are strided by 32): every rank gets whole
    groups -- at least 32 points of each group it touches -- the ranks partition the list, and the loads are balanced."""
    pts = wl.scan_points()
    owned = sharding.scan_partition(pts, world)
    assert sorted(i for o in owned for i in o) == list(range(1024))
    for o in owned:
        per_group = {}
        for i in o:
            per_group.setdefault(pts[i]["dm2_32"], 0)
            per_group[pts[i]["dm2_32"]] += 1
        assert all(c == 32 for c in per_group.values()), per_group
        assert o == sorted(o)
    sizes = [len(o) for o in owned]
    assert max(sizes) - min(sizes) <= 32
    assert owned == sharding.scan_partition(pts, world)          # deterministic


def test_scan_partition_few_groups_and_loose_points():
    one_group = [wl.table1(sin2_th23=0.3 + 0.001 * k, delta_cp=0.01 * k) for k in range(200)]
    owned = sharding.scan_partition(one_group, 4)                 # one group, four ranks: cut at multiples of 32
    assert sorted(i for o in owned for i in o) == list(range(200))
    assert all(len(o) > 0 for o in owned)
    assert sum(1 for o in owned if len(o) % 32 != 0) <= 1         # only the remainder piece is ragged
    loose = [wl.table1(dm2_32=2.0e-3 + 1e-5 * k) for k in range(10)]   # ten unrelated points
    owned = sharding.scan_partition(loose, 4)
    assert sorted(len(o) for o in owned) == [2, 2, 3, 3]
    assert sharding.scan_partition([], 2) == [[], []]
