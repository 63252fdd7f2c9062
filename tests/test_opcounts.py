"""profiles/opcounts.json, the operation counts behind bench.py's roofline fractions, must belong to the kernels that
are compiled: its SHA-256 of every kernel source has to match the tree (paper_1311_7579_b200/opcounts.py).  A kernel
edit without a new ncu capture fails here, and bench.py prints no fraction for that kernel."""
from __future__ import annotations

import os

from paper_1311_7579_b200 import opcounts


def test_counts_belong_to_the_current_kernel_sources():
    doc = opcounts.load()
    assert set(doc["kernels"]) >= {"k1", "k1b", "k2", "k4"}, "a config of bench.py has no counted kernel"
    stale = {k: opcounts.stale(k, doc) for k in doc["kernels"]}
    stale = {k: v for k, v in stale.items() if v}
    assert not stale, f"kernel sources changed since the ncu capture; re-capture and run opcounts --write: {stale}"


def test_counts_are_consistent_and_sourced():
    doc = opcounts.load()
    for key, k in doc["kernels"].items():
        assert os.path.exists(os.path.join(opcounts.ROOT, k["source"])), f"{key}: {k['source']} is not in the tree"
        assert abs(k["fp64_inst_per_unit"] - (k["dfma_per_unit"] + k["dmul_per_unit"] + k["dadd_per_unit"])) < 1e-9
        assert abs(k["flop_per_unit"] - (2 * k["dfma_per_unit"] + k["dmul_per_unit"] + k["dadd_per_unit"])) < 1e-9
        assert 0 < k["fp64_inst_per_unit"] <= k["inst_per_unit"]
        assert k["dram_bytes_per_call"] > 0
