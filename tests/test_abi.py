"""C-ABI contract checks that need no GPU: the library loads, exports every symbol include/osc.h
declares, and rejects host-checkable faults with the documented status codes.
No compute call is made here."""
from __future__ import annotations

import ctypes
import os
import re

import pytest

from paper_1311_7579_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "osc.h")

OK, INVALID, NOT_CONFIGURED, CUDA, ALIGN = 0, -1, -2, -3, -4
TABLE1 = (0.311, 0.5, 0.0251, 2.4e-3, 7.6e-5, 0.0, 2.6, 295.0, 1)


@pytest.fixture(scope="module")
def L():
    build.build_library()
    return binding.lib()


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(osc_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(L):
    names = declared_symbols()
    assert len(names) >= 22
    for name in names:
        assert hasattr(L, name), f"{name} declared in include/osc.h but not exported"
    assert set(names) == set(binding.EXPORTS)


def test_binding_has_same_names():
    import paper_1311_7579_b200 as osc

    for name in declared_symbols():
        assert callable(getattr(osc, name)), name


def test_version_and_error_string(L):
    assert b"sm_100a" in L.osc_version()
    assert isinstance(L.osc_last_error(), bytes)


def test_struct_layout_matches_header():
    # 8 doubles + int, padded to 8: the layout osc_reweight_bin_batch reads
    assert ctypes.sizeof(binding.osc_params) == 72
    assert binding.osc_params.hierarchy.offset == 64


def test_not_configured_before_set_params():
    # a fresh process: the library state is per process, so ask a child
    import subprocess
    import sys

    code = ("import ctypes;from paper_1311_7579_b200 import binding as b;L=b.lib();"
            "rc=L.osc_prob(None,0,1,1,0,None,None);print(rc, L.osc_last_error().decode())")
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, capture_output=True, text=True, check=True).stdout
    assert out.split()[0] == str(NOT_CONFIGURED), out


@pytest.mark.parametrize("idx,bad", [(0, -0.1), (0, 1.1), (1, 2.0), (2, -1e-9), (3, 0.0), (3, -2.4e-3), (4, -1e-5),
                                     (6, -1.0), (7, -5.0), (5, float("nan")), (6, float("inf")), (8, 0), (8, 2)])
def test_set_params_rejects(L, idx, bad):
    args = list(TABLE1)
    args[idx] = bad
    assert L.osc_set_params(*args) == INVALID
    assert len(L.osc_last_error()) > 0


def test_set_params_accepts_limits(L):
    assert L.osc_set_params(*TABLE1) == OK
    assert L.osc_set_params(0.0, 1.0, 0.0, 1e-3, 0.0, -3.0, 0.0, 0.0, -1) == OK
    assert L.osc_set_params(*TABLE1) == OK


def test_host_checkable_faults(L):
    assert L.osc_set_params(*TABLE1) == OK
    assert L.osc_prob(None, 0, 3, 1, 0, None, None) == INVALID      # flavour out of range
    assert L.osc_prob(None, 0, 1, -1, 0, None, None) == INVALID
    assert L.osc_prob(None, 0, 1, 1, 2, None, None) == INVALID      # antinu not 0/1
    assert L.osc_prob(None, 5, 1, 1, 0, None, None) == INVALID      # null with n > 0
    assert L.osc_prob(8, 5, 1, 1, 0, 12, None) == ALIGN             # misaligned fp64 pointer
    assert L.osc_prob(None, 0, 1, 1, 0, None, None) == OK           # n == 0 is a no-op
    assert L.osc_prob_all(None, 0, 0, None, None) == OK
    assert L.osc_prob_all(None, 3, 0, None, None) == INVALID
    assert L.osc_prob_all(None, 0, 7, None, None) == INVALID
    # osc_reweight_bin: n_bins, energy_scale, null pointers
    assert L.osc_reweight_bin(None, None, None, None, 0, 1.0, 8, 0, 8, None) == INVALID
    assert L.osc_reweight_bin(None, None, None, None, 0, 1.0, 8, 100000, 8, None) == INVALID
    assert L.osc_reweight_bin(None, None, None, None, 0, 0.0, 8, 4, 8, None) == INVALID
    assert L.osc_reweight_bin(None, None, None, None, 0, float("nan"), 8, 4, 8, None) == INVALID
    assert L.osc_reweight_bin(None, None, None, None, 0, 1.0, None, 4, 8, None) == INVALID
    assert L.osc_reweight_bin(None, None, None, None, 3, 1.0, 8, 4, 8, None) == INVALID
    assert L.osc_reweight_bin(16, 16, 16, 16, 3, 1.0, 12, 4, 8, None) == ALIGN
    # batch: bad point is reported with its index, before any launch
    pts = (binding.osc_params * 2)(binding.osc_params(*TABLE1), binding.osc_params(*TABLE1))
    pts[1].sin2_th23 = 1.5
    assert L.osc_reweight_bin_batch(pts, 2, 16, 16, 16, 16, 3, 1.0, 16, 4, 16, None) == INVALID
    assert b"point 1" in L.osc_last_error()
    assert L.osc_reweight_bin_batch(None, 2, 16, 16, 16, 16, 3, 1.0, 16, 4, 16, None) == INVALID
    assert L.osc_reweight_bin_batch(pts, -1, 16, 16, 16, 16, 3, 1.0, 16, 4, 16, None) == INVALID
    assert L.osc_get_device(None) == INVALID
    assert L.osc_fp64_peak_probe(0, 4, None, None) == INVALID
    # several energy scales in one pass: count, null list, a bad scale in the list
    sc = (ctypes.c_double * 4)(0.97, 1.0, 1.03, 1.06)
    assert L.osc_reweight_bin_scales(None, None, None, None, 0, sc, 0, 8, 4, 8, None) == INVALID
    assert L.osc_reweight_bin_scales(None, None, None, None, 0, sc, 5, 8, 4, 8, None) == INVALID
    assert L.osc_reweight_bin_scales(None, None, None, None, 0, None, 3, 8, 4, 8, None) == INVALID
    sc[1] = -1.0
    assert L.osc_reweight_bin_scales(None, None, None, None, 0, sc, 3, 8, 4, 8, None) == INVALID
    sc[1] = 1.0
    assert L.osc_reweight_bin_scales(None, None, None, None, 3, sc, 3, 8, 4, 8, None) == INVALID   # null events, n > 0
    assert L.osc_reweight_bin_scales(16, 16, 16, 16, 3, sc, 3, 12, 4, 8, None) == ALIGN
    assert L.osc_reweight_bin_scales_host(None, None, None, None, 0, sc, 0, 8, 4, 8) == INVALID
    assert L.osc_reweight_bin_scales_host(None, None, None, None, 0, None, 3, 8, 4, 8) == INVALID
    assert L.osc_reweight_bin_scales_host(None, None, None, None, 3, sc, 3, 8, 4, 8) == INVALID
    # plans: null output, bad binning, not-a-plan handles
    out = ctypes.c_void_p()
    assert L.osc_plan_create(None, None, None, None, 0, 1.0, 8, 4, None, None) == INVALID
    assert L.osc_plan_create(None, None, None, None, 0, 1.0, 8, 0, None, ctypes.byref(out)) == INVALID
    assert L.osc_plan_create(None, None, None, None, 5, 1.0, 8, 4, None, ctypes.byref(out)) == INVALID and not out.value
    junk = (ctypes.c_ulonglong * 8)()
    assert L.osc_plan_reweight_bin(None, 8, None) == INVALID
    assert L.osc_plan_reweight_bin(ctypes.addressof(junk), 8, None) == INVALID
    assert L.osc_plan_reweight_bin_batch(ctypes.addressof(junk), pts, 2, 8, None) == INVALID
    assert L.osc_plan_destroy(ctypes.addressof(junk)) == INVALID
    assert L.osc_plan_destroy(None) == OK
    # likelihood: sizes, normalisation, null pointers; no points is a no-op
    assert L.osc_neg2lnl(8, 4, 0, 8, 1.0, 8, None) == INVALID
    assert L.osc_neg2lnl(8, -1, 10, 8, 1.0, 8, None) == INVALID
    assert L.osc_neg2lnl(8, 4, 10, 8, 0.0, 8, None) == INVALID
    assert L.osc_neg2lnl(8, 4, 10, 8, float("inf"), 8, None) == INVALID
    assert L.osc_neg2lnl(None, 4, 10, 8, 1.0, 8, None) == INVALID
    assert L.osc_neg2lnl(12, 4, 10, 8, 1.0, 8, None) == ALIGN
    assert L.osc_neg2lnl(None, 0, 10, None, 1.0, None, None) == OK
    # bin-centre comparator
    assert L.osc_bin_centre_compare(None, None, None, 0, 8, 0, 8, 8, None) == INVALID          # n_bins < 1
    assert L.osc_bin_centre_compare(None, None, None, 0, 8, 4, 8, None, None) == INVALID       # null second output
    assert L.osc_bin_centre_compare(None, None, None, 3, 8, 4, 8, 8, None) == INVALID          # null events, n > 0
    assert L.osc_bin_centre_compare(16, 16, 16, 3, 8, 4, 12, 8, None) == ALIGN


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(build, "LIB_PATH", str(tmp_path / "nope.so"))
    monkeypatch.setattr(binding, "_lib", None)
    with pytest.raises(binding.OscError):
        binding.lib()


def test_binding_checks_sizes_before_handing_out_pointers():
    """Caller-supplied outputs and secondary inputs are size-checked in the binding: a short array must raise, not
    become an out-of-bounds write behind a raw pointer."""
    import numpy as np
    import torch

    e = torch.zeros(8, dtype=torch.float64)
    with pytest.raises(ValueError):
        binding.osc_prob(e, 1, 1, 0, P_out=torch.zeros(7, dtype=torch.float64))
    with pytest.raises(ValueError):
        binding.osc_prob_all(e, 0, P_out=torch.zeros(8 * 9 - 1, dtype=torch.float64))
    with pytest.raises(ValueError):
        binding.osc_bin_index(e, e, torch.zeros(8, dtype=torch.int8), 1.0, torch.zeros(3, dtype=torch.float64),
                              bin_out=torch.zeros(7, dtype=torch.int32))
    with pytest.raises(ValueError):
        binding.osc_reweight_bin(e, e, e, torch.zeros(8, dtype=torch.int8), 1.0, torch.zeros(1, dtype=torch.float64))
    h = np.zeros(8)
    ch = np.zeros(8, dtype=np.int8)
    edges = np.array([0.0, 1.0, 2.0])
    with pytest.raises(ValueError):
        binding.osc_prob_host(h, 1, 1, 0, P_out=np.zeros(7))
    with pytest.raises(ValueError):
        binding.osc_reweight_bin_host(h, h[:7], h, ch, 1.0, edges)
    with pytest.raises(ValueError):
        binding.osc_reweight_bin_host(h, h, h, ch, 1.0, edges, hist_out=np.zeros(7))
    with pytest.raises(ValueError):
        binding.osc_reweight_bin_scales_host(h, h, h, ch[:5], (1.0, 1.1), edges)
    with pytest.raises(ValueError):
        binding.osc_reweight_bin_scales_host(h, h, h, ch, (1.0, 1.1), edges, hist_out=np.zeros(8))


def test_setters_validate():
    L = binding.lib()
    assert L.osc_set_batch_path(b"k7") == INVALID and b"k7" in L.osc_last_error()
    assert L.osc_set_batch_path(b"k5") == OK and L.osc_set_batch_path(b"auto") == OK
    for path in (b"k2", b"k4", b"k4s", b"k4c"):
        assert L.osc_set_batch_path(path) == OK
    assert L.osc_set_batch_path(b"auto") == OK
    assert L.osc_set_k2_tuning(700, 0, 0, 0) == INVALID
    assert L.osc_set_k2_tuning(0, 3, 0, 0) == INVALID
    assert L.osc_set_k2_tuning(0, 0, 3, 0) == INVALID
    assert L.osc_set_k2_tuning(512, 1, 0, 0) == OK and L.osc_set_k2_tuning(0, 0, 0, 0) == OK
