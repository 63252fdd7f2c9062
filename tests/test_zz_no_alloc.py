"""osc_reweight_bin_static (include/osc.h): the fused reweight + histogram call with its scratch in a static device array,
for callers that must not allocate.  Collected last on purpose (the suite runs with pytest -x).

The test compares the new entry point with the existing path (osc_reweight_bin) on the same device arrays, two calls in
a row that differ in events, parameters, energy scale and binning -- the second call finds the first call's ticket
counters, bin-table image and partial sums in the shared array.  It passes alone in a fresh process (the static call is
then the first kernel the process launches) and after the other tests.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1311_7579_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RTOL = 1e-12          # the tolerance the tests use between two GPU paths (test_parity_gpu.py: plans, chunked host calls)


@pytest.fixture(scope="module")
def osc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1311_7579_b200 import build

    build.build_library()
    import paper_1311_7579_b200 as m

    torch.cuda.set_device(0)
    m.osc_set_device(0)
    return m


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


CASES = [
    # events, seed, parameters, energy scale, bin edges
    (300_000 + 7, 71, wl.table1(), 1.0, wl.bin_edges()),
    (1_000_000 + 1, 72, wl.table1(delta_cp=-1.3, rho_g_cm3=5.0, L_km=1300.0, hierarchy=-1), 0.97, wl.bin_edges(128, 6.0)),
]


def test_static_scratch_call_equals_the_existing_path_on_two_calls_in_a_row(osc):
    # every STATIC call first, back to back, so that the second one starts from what the first one left in the array
    inputs, got = [], []
    for n, seed, par, scale, edges in CASES:
        et, er, w0, ch = wl.events(n, seed=seed)
        et[11] = float("nan"); ch[12] = 9; er[13] = -1.0                    # dropped events
        d = [dev(a) for a in (et, er, w0, ch)]
        de = dev(edges)
        out = torch.full((osc.N_CHANNELS, len(edges) - 1), -7.0, dtype=torch.float64, device="cuda")   # must be overwritten
        osc.osc_set_params(**par)
        osc.osc_reweight_bin_static(*d, scale, de, out)
        inputs.append((d, de, (et, er, w0, ch)))
        got.append(out)
    torch.cuda.synchronize()
    for (n, seed, par, scale, edges), (d, de, h), out in zip(CASES, inputs, got):
        osc.osc_set_params(**par)
        ref = osc.osc_reweight_bin(*d, scale, de).cpu().numpy()
        a = out.cpu().numpy()
        assert np.all(np.isfinite(a)) and np.all(a[ref == 0.0] == 0.0)
        np.testing.assert_allclose(a, ref, rtol=RTOL, atol=0.0)
        # same call again: the shared array now holds this call's own leftovers; bit-reproducible
        again = torch.empty_like(out)
        osc.osc_reweight_bin_static(*d, scale, de, again)
        assert np.array_equal(again.cpu().numpy(), a)
    # and against the oracle (1e-9 per bin, the bar of the parity tests) on the first case
    (n, seed, par, scale, edges), (_, _, (et, er, w0, ch)) = CASES[0], inputs[0]
    want = oracle.reweight_bin(oracle.Params(**par), et, er, w0, ch, scale, edges)
    a = got[0].cpu().numpy()
    err = np.abs(a - want)
    assert np.all(err <= 1e-9 * np.maximum(np.abs(want), 1e-14)), float(err.max())


def test_static_scratch_call_sizes_and_limits(osc):
    osc.osc_set_params(**wl.table1())
    et, er, w0, ch = wl.events(1000, seed=73)
    d = [dev(a) for a in (et, er, w0, ch)]
    # n = 0: hist_out is zeroed
    out = torch.full((osc.N_CHANNELS, 50), 3.0, dtype=torch.float64, device="cuda")
    osc.osc_reweight_bin_static(*[t[:0] for t in d], 1.0, dev(wl.bin_edges()), out)
    assert float(out.abs().sum()) == 0.0
    # small and ragged n
    for n in (1, 33, 1000):
        sub = [t[:n] for t in d]
        osc.osc_reweight_bin_static(*sub, 1.03, dev(wl.bin_edges()), out)
        ref = osc.osc_reweight_bin(*sub, 1.03, dev(wl.bin_edges()))
        np.testing.assert_allclose(out.cpu().numpy(), ref.cpu().numpy(), rtol=RTOL, atol=0.0)
    # beyond the stated maximum: a clear error, nothing launched, the output untouched
    edges = dev(wl.bin_edges(129, 5.0))
    big = torch.full((osc.N_CHANNELS, 129), 5.0, dtype=torch.float64, device="cuda")
    with pytest.raises(osc.OscError) as ei:
        osc.osc_reweight_bin_static(*d, 1.0, edges, big)
    assert "128" in str(ei.value) and "osc_reweight_bin_static" in str(ei.value)
    torch.cuda.synchronize()
    assert float((big - 5.0).abs().sum()) == 0.0


def test_static_scratch_call_under_stream_capture(osc):
    """What the entry point is for: the call is captured into a CUDA graph (a cudaMalloc inside the capture would
    invalidate it) and replayed on new contents of the same buffers."""
    n, edges = 200_000, wl.bin_edges()
    osc.osc_set_params(**wl.table1())
    d = [dev(a) for a in wl.events(n, seed=74)]
    de = dev(edges)
    out = torch.zeros((osc.N_CHANNELS, len(edges) - 1), dtype=torch.float64, device="cuda")
    osc.osc_reweight_bin_static(*d, 1.0, de, out)              # set-up outside the capture: symbol address, attributes
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.graph(g, stream=side):
        osc.osc_reweight_bin_static(*d, 1.0, de, out, stream=torch.cuda.current_stream())
    for seed in (75, 76):
        fresh = wl.events(n, seed=seed)
        for t_dev, a in zip(d, fresh):
            t_dev.copy_(torch.from_numpy(np.ascontiguousarray(a)))
        out.fill_(-1.0)
        g.replay()
        torch.cuda.synchronize()
        ref = osc.osc_reweight_bin(*d, 1.0, de).cpu().numpy()
        np.testing.assert_allclose(out.cpu().numpy(), ref, rtol=RTOL, atol=0.0)
