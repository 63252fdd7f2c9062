"""GPU-vs-oracle parity (SURVEY.md section 4 tier T2/T3/T4), through the C ABI, on a B200.

Bars (BASELINE.json:north_star): every fp64 probability within 1e-10 absolute of the oracle, every
fp64 histogram bin within 1e-9 relative, integer bin indices bit-exact.  Inputs are the seeded arrays
of paper_1311_7579_b200.workloads, handed byte-identical to both sides.  No expected value here comes
from the CUDA path.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle
from paper_1311_7579_b200 import workloads as wl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

P_ABS = 1e-10     # north_star: absolute, per probability
H_REL = 1e-9      # north_star: relative, per histogram bin
H_ZERO = 1e-25    # see assert_hist_close


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


def host(t):
    return t.cpu().numpy()


def assert_prob_close(got, ref, what=""):
    assert got.shape == ref.shape
    assert np.array_equal(np.isnan(got), np.isnan(ref)), f"{what}: NaN pattern differs"
    m = ~np.isnan(ref)
    err = float(np.max(np.abs(got[m] - ref[m]))) if m.any() else 0.0
    assert err <= P_ABS, f"{what}: max |dP| = {err:.3e} > {P_ABS}"
    return err


def assert_hist_close(got, ref, what=""):
    """1e-9 relative on every bin.  Bins no event falls into are exactly 0.0 on both sides.  H_ZERO keeps the
    relative bar meaningful where the probability itself is a computed zero (e.g. P(numu->nue) at L = 0: the
    oracle's long-double rounding leaves ~1e-39 where the closed form gives exactly 0): it is 25 orders below
    any event weight of these workloads."""
    assert got.shape == ref.shape
    assert np.all(got[ref == 0.0] == 0.0), f"{what}: a bin the oracle leaves empty is not 0.0"
    assert np.all(np.isfinite(got)), f"{what}: non-finite bin"
    err = np.abs(got - ref)
    bad = err > H_REL * np.abs(ref) + H_ZERO
    nz = np.abs(ref) > H_ZERO
    rel = float(np.max(err[nz] / np.abs(ref[nz]))) if nz.any() else 0.0
    assert not bad.any(), f"{what}: max rel bin error {rel:.3e} > {H_REL}"
    return rel


def set_params(osc, par):
    osc.osc_set_params(**par)
    return oracle.Params(**par)


# ------------------------------------------------------------------------------------------------
# configs[0]: 1e5 events, Table 1, P(numu->numu) and P(numu->nue)
# ------------------------------------------------------------------------------------------------
def test_config0(osc):
    E = wl.e_true(100_000, seed=0)
    op = set_params(osc, wl.table1())
    dE = dev(E)
    for fin, fout in ((1, 1), (1, 0)):
        got = host(osc.osc_prob(dE, fin, fout, 0))
        assert_prob_close(got, oracle.prob(op, E, fin, fout, 0), f"config0 {fin}->{fout}")


# ------------------------------------------------------------------------------------------------
# configs[1] at a size the oracle finishes in seconds: all 9 transitions x nu/nubar, 4 delta draws x
# both hierarchies; several tiles and a ragged tail
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("run", range(8))
def test_config1_all_transitions(osc, run):
    par = wl.config1_runs()[run]
    n = 40_000 + 2 * 256 * 3 + 131
    E = wl.e_true(n, seed=1)
    op = set_params(osc, par)
    dE = dev(E)
    for anti in (0, 1):
        got = host(osc.osc_prob_all(dE, anti))
        assert_prob_close(got, oracle.prob_all(op, E, anti), f"config1 run {run} anti {anti}")
        assert got.min() >= 0.0      # (unitarity: test_unitarity_through_nine_independent_calls)


def test_single_transition_equals_all(osc):
    par = wl.config1_runs()[3]
    E = wl.e_true(6_001, seed=11)
    op = set_params(osc, par)
    dE = dev(E)
    for anti in (0, 1):
        ref = oracle.prob_all(op, E, anti)
        for a in range(3):
            for b in range(3):
                got = host(osc.osc_prob(dE, a, b, anti))
                assert_prob_close(got, ref[3 * b + a], f"{a}->{b} anti {anti}")


# ------------------------------------------------------------------------------------------------
# configs[4] parameter settings: rho x L x hierarchy, and harder corners (degenerate spectra, L = 0,
# large density, resonance)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", range(12))
def test_sweep_settings_prob(osc, k):
    par = wl.sweep_settings()[k]
    E = wl.e_true(20_000, seed=40 + k)
    op = set_params(osc, par)
    dE = dev(E)
    for anti in (0, 1):
        assert_prob_close(host(osc.osc_prob_all(dE, anti)), oracle.prob_all(op, E, anti), f"sweep {k} anti {anti}")


CORNERS = [
    dict(rho_g_cm3=0.0, dm2_21=0.0, sin2_th13=0.0),               # exactly degenerate pair in vacuum (P3)
    dict(rho_g_cm3=2.6, dm2_21=0.0, sin2_th13=0.0),               # degenerate pair in matter
    dict(rho_g_cm3=2.6, dm2_21=0.0),                              # one mass scale (P7)
    dict(rho_g_cm3=2.6, sin2_th13=0.0),                           # solar sector only (P8)
    dict(L_km=0.0),                                               # P = delta (P5)
    dict(rho_g_cm3=50.0, L_km=1300.0),                            # large density
    dict(rho_g_cm3=100.0, L_km=2000.0, hierarchy=-1),
    dict(rho_g_cm3=12.0, L_km=1300.0, delta_cp=1.3),              # atmospheric resonance inside 0.1-10 GeV
    dict(sin2_th12=0.0, sin2_th13=0.0, sin2_th23=0.0),            # U = 1
    dict(sin2_th12=1.0, sin2_th13=1.0, sin2_th23=1.0, delta_cp=-2.0),
    dict(sin2_th23=0.3, delta_cp=-math.pi / 2, hierarchy=-1, L_km=1300.0),
    dict(dm2_32=1e-3, dm2_21=9.9e-4, delta_cp=2.5),               # comparable splittings
    dict(dm2_32=2.4e-3, dm2_21=2.4e-3, hierarchy=-1),             # inverted: dm2_31 = 0 -> m1 = m3 degenerate
]


@pytest.mark.parametrize("k", range(len(CORNERS)))
def test_corner_parameters(osc, k):
    par = wl.table1(**CORNERS[k])
    E = np.concatenate([wl.e_true(5_000, seed=60 + k), np.geomspace(0.1, 10.0, 1_237)])
    op = set_params(osc, par)
    dE = dev(E)
    for anti in (0, 1):
        assert_prob_close(host(osc.osc_prob_all(dE, anti)), oracle.prob_all(op, E, anti), f"corner {k} anti {anti}")
        for fin, fout in ((1, 1), (1, 0), (0, 0), (2, 1)):
            assert_prob_close(host(osc.osc_prob(dE, fin, fout, anti)), oracle.prob(op, E, fin, fout, anti),
                              f"corner {k} {fin}->{fout} anti {anti}")


def test_random_parameter_sets(osc):
    rng = np.random.Generator(np.random.PCG64(77))
    E = np.concatenate([wl.e_true(1_500, seed=78), np.geomspace(0.1, 10.0, 500)])
    dE = dev(E)
    worst = 0.0
    for _ in range(60):
        par = dict(sin2_th12=rng.uniform(0, 1), sin2_th23=rng.uniform(0, 1), sin2_th13=rng.uniform(0, 1),
                   dm2_32=10 ** rng.uniform(-4, -2), dm2_21=10 ** rng.uniform(-6, -3),
                   delta_cp=rng.uniform(-math.pi, math.pi), rho_g_cm3=rng.uniform(0, 15),
                   L_km=rng.uniform(0, 2000), hierarchy=int(rng.choice([1, -1])))
        op = set_params(osc, par)
        for anti in (0, 1):
            worst = max(worst, assert_prob_close(host(osc.osc_prob_all(dE, anti)), oracle.prob_all(op, E, anti),
                                                 f"random {par} anti {anti}"))
    print(f"random parameter sets: worst |dP| = {worst:.3e}")


# ------------------------------------------------------------------------------------------------
# A11: unusable energies, ragged sizes, unaligned slices
# ------------------------------------------------------------------------------------------------
def test_bad_energies_give_nan(osc):
    op = set_params(osc, wl.table1())
    E = wl.e_true(1_031, seed=5)
    E[[0, 7, 512, 513, 1030]] = [0.0, -1.0, np.nan, np.inf, -np.inf]
    E[100] = -0.0
    dE = dev(E)
    assert_prob_close(host(osc.osc_prob(dE, 1, 0, 0)), oracle.prob(op, E, 1, 0, 0), "bad energies")
    assert_prob_close(host(osc.osc_prob_all(dE, 1)), oracle.prob_all(op, E, 1), "bad energies all")


@pytest.mark.parametrize("n", [1, 2, 3, 31, 32, 33, 255, 256, 257, 511, 512, 513, 1023, 1025, 4097])
def test_ragged_sizes(osc, n):
    op = set_params(osc, wl.table1(delta_cp=0.7))
    E = wl.e_true(n + 1, seed=n)
    d = dev(E)
    for off in (0, 1):                      # off = 1: 8-byte aligned only -> scalar path
        Es = E[off:off + n]
        o0 = 2 - off                        # off = 0: output 16-byte aligned too -> 128-bit path
        out = torch.full((n + 4,), -7.0, dtype=torch.float64, device="cuda")
        osc.osc_prob(d[off:off + n], 1, 1, 0, P_out=out[o0:o0 + n])
        o = host(out)
        assert np.all(o[:o0] == -7.0) and np.all(o[o0 + n:] == -7.0), "wrote outside P_out"
        assert_prob_close(o[o0:o0 + n], oracle.prob(op, Es, 1, 1, 0), f"ragged n={n} off={off}")
        pa = torch.full((9 * n + 2,), -7.0, dtype=torch.float64, device="cuda")
        osc.osc_prob_all(d[off:off + n], 0, P_out=pa[1:1 + 9 * n])
        o = host(pa)
        assert o[0] == -7.0 and o[-1] == -7.0
        assert_prob_close(o[1:1 + 9 * n].reshape(9, n), oracle.prob_all(op, Es, 0), f"ragged all n={n}")


def test_ragged_sizes_wide_blocks(osc):
    """osc_prob above ~4.5e5 events runs as one block of 768 threads per SM: the three assemblies (e->e, another
    diagonal element, off-diagonal), 128-bit and scalar path, a ragged tail, and nothing written outside P_out."""
    n = 2 * 148 * 768 * 2 + 768 * 2 * 3 + 5
    op = set_params(osc, wl.table1(delta_cp=-0.4))
    E = wl.e_true(n + 1, seed=4242)
    E[[11, n // 2, n - 1]] = [np.nan, 0.0, -2.0]
    d = dev(E)
    worst = 0.0
    for off in (0, 1):
        Es = E[off:off + n]
        o0 = 2 - off
        for fin, fout, anti in ((0, 0, 0), (1, 1, 1), (1, 0, 0)):
            out = torch.full((n + 4,), -7.0, dtype=torch.float64, device="cuda")
            osc.osc_prob(d[off:off + n], fin, fout, anti, P_out=out[o0:o0 + n])
            o = host(out)
            assert np.all(o[:o0] == -7.0) and np.all(o[o0 + n:] == -7.0), "wrote outside P_out"
            worst = max(worst, assert_prob_close(o[o0:o0 + n], oracle.prob(op, Es, fin, fout, anti),
                                                 f"wide blocks {fin}->{fout} off={off}"))
    print(f"wide blocks: worst |dP| = {worst:.3e}")


def test_n_zero(osc):
    set_params(osc, wl.table1())
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    assert osc.osc_prob(e, 1, 1, 0).numel() == 0
    assert osc.osc_prob_all(e, 0).numel() == 0
    edges = dev(wl.bin_edges())
    h = torch.full((4, 50), 3.0, dtype=torch.float64, device="cuda")
    osc.osc_reweight_bin(e, e, e, torch.empty(0, dtype=torch.int8, device="cuda"), 1.0, edges, hist_out=h)
    assert float(h.abs().sum()) == 0.0      # overwritten (zeroed) even with no events
    hb = torch.full((2, 4, 50), 3.0, dtype=torch.float64, device="cuda")
    osc.osc_reweight_bin_batch([wl.table1(), wl.table1()], e, e, e, torch.empty(0, dtype=torch.int8, device="cuda"),
                               1.0, edges, hist_out=hb)
    assert float(hb.abs().sum()) == 0.0


# ------------------------------------------------------------------------------------------------
# configs[2]: fused reweight + histogram; bin indices bit-exact
# ------------------------------------------------------------------------------------------------
def test_config2_histograms(osc):
    n = 300_000 + 2 * 256 * 5 + 77
    et, er, w0, ch = wl.events(n, seed=2)
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1())
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    for s in wl.ENERGY_SCALES:
        got = host(osc.osc_reweight_bin(*d, s, de))
        ref = oracle.reweight_bin(op, et, er, w0, ch, s, edges)
        assert_hist_close(got, ref, f"config2 s={s}")
        bi = host(osc.osc_bin_index(d[0], d[1], d[3], s, de))
        assert np.array_equal(bi, oracle.bin_index(et, er, ch, s, edges)), f"bin indices differ at s={s}"


@pytest.mark.parametrize("k", range(12))
def test_sweep_settings_histograms(osc, k):
    par = wl.sweep_settings()[k]
    n = 50_000 + k
    et, er, w0, ch = wl.events(n, seed=100 + k)
    edges = wl.bin_edges()
    op = set_params(osc, par)
    got = host(osc.osc_reweight_bin(dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
    assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, 1.0, edges), f"sweep hist {k}")


def test_bin_index_bit_exact_large_and_edges(osc):
    n = 1_000_000
    et, er, w0, ch = wl.events(n, seed=7)
    edges = wl.bin_edges()
    # events exactly on edges (upper bin), just below, on the last edge (dropped), negative, NaN, -0.0
    er[:51] = edges
    er[51:102] = np.nextafter(edges, -np.inf)
    er[102:153] = np.nextafter(edges, np.inf)
    er[153:158] = [np.nan, -0.0, np.inf, -np.inf, -1e-300]
    et[200:204] = [0.0, -3.0, np.nan, np.inf]
    ch[300:304] = [-1, 4, 127, -128]
    set_params(osc, wl.table1())
    d_et, d_er, d_ch, de = dev(et), dev(er), dev(ch), dev(edges)
    for s in (0.97, 1.0, 1.03, 1.0 / 3.0, 7.123456789):
        bi = host(osc.osc_bin_index(d_et, d_er, d_ch, s, de))
        assert np.array_equal(bi, oracle.bin_index(et, er, ch, s, edges)), f"s={s}"


def test_dropped_and_bad_events_are_skipped(osc):
    n = 20_011
    et, er, w0, ch = wl.events(n, seed=8)
    edges = wl.bin_edges()
    er[:51] = edges
    er[60:63] = [np.nan, -1.0, 1e9]
    et[100:104] = [0.0, -3.0, np.nan, np.inf]
    ch[300:304] = [-1, 4, 127, -128]
    w0[500] = 0.0
    op = set_params(osc, wl.table1(delta_cp=-1.0))
    got = host(osc.osc_reweight_bin(dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
    assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, 1.0, edges), "bad events")


@pytest.mark.parametrize("threads", [256, 384, 512])
@pytest.mark.parametrize("nb", [1, 7, 50])
def test_one_sub_histogram_per_warp_under_collisions(osc, nb, threads):
    """The layout of large binnings (one sub-histogram per warp for both events of a lane), forced onto few bins so that
    most lanes of a warp, and both events of a lane, hit the same word: every weight must still arrive exactly once."""
    n = 60_013
    et, er, w0, ch = wl.events(n, seed=31 + nb)
    er[:n // 3] = 0.7                                   # one third of all events in one bin
    edges = wl.bin_edges(nb, 5.0)
    op = set_params(osc, wl.table1())
    ref = oracle.reweight_bin(op, et, er, w0, ch, 1.0, edges)
    osc.osc_set_k2_tuning(threads=threads, slots=1)
    try:
        for off in (0, 1):                                  # 128-bit and scalar loads
            got = host(osc.osc_reweight_bin(dev(et)[off:], dev(er)[off:], dev(w0)[off:], dev(ch)[off:], 1.0, dev(edges)))
            want = ref if off == 0 else oracle.reweight_bin(op, et[1:], er[1:], w0[1:], ch[1:], 1.0, edges)
            assert_hist_close(got, want, f"single slot, {nb} bins, {threads} threads, off={off}")
            again = host(osc.osc_reweight_bin(dev(et)[off:], dev(er)[off:], dev(w0)[off:], dev(ch)[off:], 1.0, dev(edges)))
            assert np.array_equal(got, again), "not bit-reproducible"
    finally:
        osc.osc_set_k2_tuning()


@pytest.mark.parametrize("nb,kind", [(1, "uniform"), (2, "uniform"), (3, "log"), (7, "random"), (50, "random"),
                                     (64, "uniform"), (140, "uniform"), (141, "random"), (200, "log"),
                                     (210, "uniform"), (215, "random"), (250, "uniform"), (290, "log"),
                                     (425, "uniform"), (430, "random"), (570, "uniform"), (575, "log"),
                                     (768, "uniform")])
def test_bin_layouts(osc, nb, kind):
    n = 30_007
    et, er, w0, ch = wl.events(n, seed=9)
    rng = np.random.Generator(np.random.PCG64(nb))
    if kind == "uniform":
        edges = wl.bin_edges(nb, 5.0)
    elif kind == "log":
        edges = np.geomspace(0.05, 6.0, nb + 1)
    else:
        edges = np.sort(rng.uniform(-0.5, 5.0, nb + 1))
        assert np.all(np.diff(edges) > 0)
    op = set_params(osc, wl.table1())
    d_et, d_er, d_w, d_ch, de = dev(et), dev(er), dev(w0), dev(ch), dev(edges)
    got = host(osc.osc_reweight_bin(d_et, d_er, d_w, d_ch, 1.03, de))
    assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, 1.03, edges), f"nb={nb} {kind}")
    assert np.array_equal(host(osc.osc_bin_index(d_et, d_er, d_ch, 1.03, de)),
                          oracle.bin_index(et, er, ch, 1.03, edges))


@pytest.mark.parametrize("n", [1, 2, 31, 33, 511, 513, 1025, 5000])
def test_histogram_ragged_and_unaligned(osc, n):
    et, er, w0, ch = wl.events(n + 1, seed=300 + n)
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1())
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    for off in (0, 1):
        got = host(osc.osc_reweight_bin(*[t[off:off + n] for t in d], 1.0, de))
        ref = oracle.reweight_bin(op, *[a[off:off + n] for a in (et, er, w0, ch)], 1.0, edges)
        assert_hist_close(got, ref, f"n={n} off={off}")


def test_histogram_is_bit_reproducible(osc):
    n = 400_003
    et, er, w0, ch = wl.events(n, seed=10)
    set_params(osc, wl.table1())
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(wl.bin_edges())
    a = host(osc.osc_reweight_bin(*d, 1.0, de))
    for _ in range(3):
        assert np.array_equal(a, host(osc.osc_reweight_bin(*d, 1.0, de)))


# ------------------------------------------------------------------------------------------------
# configs[3]: batched parameter scan
# ------------------------------------------------------------------------------------------------
def test_config3_full_grid_small_sample(osc):
    pts = wl.scan_points()
    assert len(pts) == 1024
    n = 2_003
    et, er, w0, ch = wl.events(n, seed=3)
    edges = wl.bin_edges()
    got = host(osc.osc_reweight_bin_batch(pts, dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    assert got.shape == (1024, 4, 50)
    assert_hist_close(got, ref, "config3 grid")


def test_config3_diagonal_more_events(osc):
    pts = wl.scan_points()[::33][:16]
    n = 60_000 + 19
    et, er, w0, ch = wl.events(n, seed=3)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    got = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    assert_hist_close(got, ref, "config3 diagonal")


def test_batch_point_count_edge_cases(osc):
    n = 5_003
    et, er, w0, ch = wl.events(n, seed=12)
    edges = wl.bin_edges(13, 4.0)
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    mixed = [wl.table1(), wl.table1(hierarchy=-1, rho_g_cm3=0.0), wl.table1(L_km=1300.0, delta_cp=2.0),
             wl.table1(sin2_th13=0.0, dm2_21=0.0), wl.table1(L_km=0.0)]
    for npts in (1, 2, 5):
        pts = mixed[:npts]
        got = host(osc.osc_reweight_bin_batch(pts, *d, 0.97, de))
        ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 0.97, edges)
        assert_hist_close(got, ref, f"batch npts={npts}")
    # the batched call does not depend on, and does not change, the osc_set_params state
    op = set_params(osc, wl.table1(delta_cp=0.4))
    osc.osc_reweight_bin_batch(mixed, *d, 1.0, de)
    got = host(osc.osc_reweight_bin(*d, 1.0, de))
    assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, 1.0, edges), "state after batch")


# ------------------------------------------------------------------------------------------------
# k4, the factorised path of the batched call (points that differ only in theta23 / delta_cp share the
# eigen-problem).  osc_set_batch_path forces one path or the other (include/osc.h), so both are checked against the
# oracle on the same inputs, and against each other.  k4 has two main kernels: "k4s" (shared-memory slice, lane = point)
# and "k4c" (one launch per sub-group, monomials in the kernel parameters, lane = event); "k4" lets the library choose
# (k4c from 1e5 events on).
# ------------------------------------------------------------------------------------------------
K4_PATHS = ["k4s", "k4c"]


class batch_path:
    def __init__(self, which):
        self.which = which

    def __enter__(self):
        import paper_1311_7579_b200 as m
        m.osc_set_batch_path(self.which)

    def __exit__(self, *a):
        import paper_1311_7579_b200 as m
        m.osc_set_batch_path("auto")


def ragged_group_points(seed=21):
    """Three eigen-problems with 1, 33 and 36 points (the second and third spill into a second sub-group of lanes),
    interleaved in the list; theta23 covers 0 and 1, delta_cp the whole circle."""
    rng = np.random.default_rng(seed)
    bases = [wl.table1(rho_g_cm3=0.0, L_km=1300.0, hierarchy=-1),
             wl.table1(dm2_32=2.1e-3, rho_g_cm3=5.0),
             wl.table1(sin2_th13=0.03, sin2_th12=0.28, L_km=810.0)]
    sizes = [1, 33, 36]
    pts = []
    for g, (b, m) in enumerate(zip(bases, sizes)):
        th = rng.uniform(0.0, 1.0, m)
        th[0] = 0.0 if g == 1 else th[0]
        th[-1] = 1.0 if g == 2 else th[-1]
        for k in range(m):
            pts.append(dict(b, sin2_th23=float(th[k]), delta_cp=float(rng.uniform(-math.pi, math.pi))))
    order = rng.permutation(len(pts))
    return [pts[i] for i in order]


def test_k4_ragged_groups_vs_oracle(osc):
    pts = ragged_group_points()
    n = 3_000 + 7
    et, er, w0, ch = wl.events(n, seed=22)
    et[5] = -1.0; et[6] = float("nan"); ch[7] = 9; ch[8] = -3; er[9] = 77.0     # dropped events (A8, A11)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.03, edges)
    got4 = {}
    for path in K4_PATHS:
        with batch_path(path):
            got4[path] = host(osc.osc_reweight_bin_batch(pts, *d, 1.03, dev(edges)))
    with batch_path("k2"):
        got3 = host(osc.osc_reweight_bin_batch(pts, *d, 1.03, dev(edges)))
    with batch_path("k5"):
        got5 = host(osc.osc_reweight_bin_batch(pts, *d, 1.03, dev(edges)))
    for path in K4_PATHS:
        assert_hist_close(got4[path], ref, f"{path} ragged groups")
        assert np.array_equal(got4[path] == 0.0, got3 == 0.0)
    assert_hist_close(got3, ref, "k2-per-point ragged groups")
    assert_hist_close(got5, ref, "k5 ragged groups")
    assert np.array_equal(got5 == 0.0, got3 == 0.0)


@pytest.mark.parametrize("k4", K4_PATHS)
def test_k4_equals_k3_on_the_grid_with_more_events(osc, k4):
    pts = wl.scan_points()[:96]          # three dm2_32 groups of 32 points
    n = 200_000 + 33
    et, er, w0, ch = wl.events(n, seed=23)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    with batch_path(k4):
        a = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
        b = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
    with batch_path("k2"):
        c = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
    with batch_path("k5"):
        e = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
        f = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
    assert np.array_equal(a, b), "k4 is not bit-reproducible"
    assert np.array_equal(e, f), "k5 is not bit-reproducible"
    assert_hist_close(a, c, "k4 vs k2 per point")
    assert_hist_close(e, c, "k5 vs k2 per point")
    # the oracle on a sample of points (full 200k events each)
    pick = [0, 37, 95]
    ref = oracle.reweight_bin_batch([oracle.Params(**pts[i]) for i in pick], et, er, w0, ch, 1.0, edges)
    assert_hist_close(a[pick], ref, "k4 vs oracle")


@pytest.mark.parametrize("path", K4_PATHS + ["k5"])
@pytest.mark.parametrize("n", [0, 1, 31, 64, 65, 129, 1000])
@pytest.mark.parametrize("nb,kind", [(1, "uniform"), (7, "random"), (50, "uniform")])
def test_k4_small_and_ragged_sizes(osc, n, nb, kind, path):
    rng = np.random.default_rng(100 + n + nb)
    if kind == "uniform":
        edges = wl.bin_edges(nb, 5.0)
    else:
        edges = np.sort(rng.uniform(0.05, 6.0, nb + 1))
    pts = [wl.table1(sin2_th23=0.3 + 0.05 * k, delta_cp=-3.0 + 0.7 * k) for k in range(9)]
    et, er, w0, ch = wl.events(max(n, 1), seed=24)
    et, er, w0, ch = et[:n], er[:n], w0[:n], ch[:n]
    with batch_path(path):
        got = host(osc.osc_reweight_bin_batch(pts, dev(et), dev(er), dev(w0), dev(ch), 0.97, dev(edges)))
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 0.97, edges)
    assert got.shape == (9, 4, nb)
    assert_hist_close(got, ref, f"{path} n={n} nb={nb}")


@pytest.mark.parametrize("path", ["k2"] + K4_PATHS + ["k5"])
def test_batch_paths_with_many_bins(osc, path):
    """350 bins x 4 channels = 1400 cells: the per-warp counters of the sort passes and the cell search of the piece
    kernels at a size well beyond configs[3]'s 200 cells; "k2" is one pass of the single-set kernel per point."""
    n = 30_000 + 5
    et, er, w0, ch = wl.events(n, seed=26)
    edges = wl.bin_edges(350, 5.0)
    pts = [wl.table1(sin2_th23=0.35 + 0.02 * k, delta_cp=-2.0 + 0.3 * k) for k in range(12)]
    with batch_path(path):
        got = host(osc.osc_reweight_bin_batch(pts, dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    assert_hist_close(got, ref, f"{path} with 350 bins")


def test_batch_sorted_paths_with_768_bins(osc):
    """The largest binning the library accepts (768 bins, 3072 cells): only the sorted paths take it in a batch."""
    n = 10_000
    et, er, w0, ch = wl.events(n, seed=27)
    edges = wl.bin_edges(768, 5.0)
    pts = [wl.table1(sin2_th23=0.3 + 0.04 * k, dm2_32=2.2e-3 + 1e-5 * (k // 5)) for k in range(10)]
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    for path in K4_PATHS + ["k5"]:
        with batch_path(path):
            got = host(osc.osc_reweight_bin_batch(pts, dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
        assert_hist_close(got, ref, f"{path} with 768 bins")


@pytest.mark.parametrize("path", K4_PATHS + ["k5"])
def test_batch_sorted_paths_on_corner_parameters(osc, path):
    """The degenerate and extreme parameter sets of test_corner_parameters through the sorted batched kernels: every
    corner as its own group (k5), and every corner with four (theta23, delta) variations (k4)."""
    n = 6_000 + 1
    et, er, w0, ch = wl.events(n, seed=28)
    edges = wl.bin_edges()
    pts = []
    for c in CORNERS:
        base = wl.table1(**c)
        for k in range(4 if path in K4_PATHS else 1):
            pts.append(dict(base, sin2_th23=base["sin2_th23"] if k == 0 else 0.2 + 0.2 * k,
                            delta_cp=base["delta_cp"] if k == 0 else -2.5 + 1.7 * k))
    with batch_path(path):
        got = host(osc.osc_reweight_bin_batch(pts, dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    assert_hist_close(got, ref, f"{path} on corner parameters")


def test_batch_keeps_the_plan_of_the_last_point_list_only_while_it_is_the_same(osc):
    """The library keeps the host-side plan of the last point list (compared bytewise): a repeated list must give the same
    histograms, a list of the same length that differs in one number must give its own."""
    n = 20_000 + 3
    et, er, w0, ch = wl.events(n, seed=29)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    a_pts = [wl.table1(sin2_th23=0.35 + 0.01 * k, delta_cp=-1.0 + 0.1 * k) for k in range(16)]
    b_pts = [dict(q) for q in a_pts]
    b_pts[7]["delta_cp"] = 2.5                        # same group structure, one monomial set differs
    c_pts = [dict(q) for q in a_pts]
    c_pts[3]["dm2_32"] = 2.7e-3                       # one point leaves the group
    for path in K4_PATHS + ["k5"]:
        with batch_path(path):
            a1 = host(osc.osc_reweight_bin_batch(a_pts, *d, 1.0, de))
            b1 = host(osc.osc_reweight_bin_batch(b_pts, *d, 1.0, de))
            a2 = host(osc.osc_reweight_bin_batch(a_pts, *d, 1.0, de))
            a3 = host(osc.osc_reweight_bin_batch(a_pts, *d, 1.0, de))
            c1 = host(osc.osc_reweight_bin_batch(c_pts, *d, 1.0, de))
        assert np.array_equal(a1, a2) and np.array_equal(a2, a3), path
        for name, pts, got in (("a", a_pts, a1), ("b", b_pts, b1), ("c", c_pts, c1)):
            ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
            assert_hist_close(got, ref, f"{path}, list {name}")
        assert not np.array_equal(a1[7], b1[7]) and np.array_equal(a1[6], b1[6])


@pytest.mark.parametrize("k4", K4_PATHS)
def test_k4_all_events_dropped(osc, k4):
    n = 500
    et, er, w0, ch = wl.events(n, seed=25)
    er[:] = 99.0
    pts = [wl.table1(sin2_th23=0.4), wl.table1(sin2_th23=0.6)]
    with batch_path(k4):
        got = host(osc.osc_reweight_bin_batch(pts, dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(wl.bin_edges())))
    assert got.shape == (2, 4, 50) and float(np.abs(got).sum()) == 0.0


# ------------------------------------------------------------------------------------------------
# NEXT-3: several energy scales in one pass (osc_reweight_bin_scales)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("scales", [(1.0,), (0.97, 1.03), wl.ENERGY_SCALES, (0.9, 0.97, 1.0, 1.1)])
def test_scales_one_pass_vs_oracle_and_single_calls(osc, scales):
    n = 300_000 + 11
    et, er, w0, ch = wl.events(n, seed=41)
    et[3] = 0.0; ch[4] = 7; er[5] = -2.0
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    op = set_params(osc, wl.table1(delta_cp=-1.1))
    got = host(osc.osc_reweight_bin_scales(*d, scales, de))
    again = host(osc.osc_reweight_bin_scales(*d, scales, de))
    assert got.shape == (len(scales), 4, 50) and np.array_equal(got, again)
    for k, s in enumerate(scales):
        assert_hist_close(got[k], oracle.reweight_bin(op, et, er, w0, ch, s, edges), f"scales[{k}]={s}")
        single = host(osc.osc_reweight_bin(*d, s, de))
        np.testing.assert_allclose(got[k], single, rtol=1e-12, atol=0.0)


@pytest.mark.parametrize("n", [0, 1, 33, 513, 1025])
def test_scales_ragged_and_unaligned(osc, n):
    et, er, w0, ch = wl.events(n + 3, seed=42)
    edges = wl.bin_edges(13, 4.0)
    op = set_params(osc, wl.table1(hierarchy=-1))
    big = [dev(a) for a in (et, er, w0, ch)]
    d = [t[1:1 + n] for t in big]                      # 8-byte aligned only: the scalar load path
    got = host(osc.osc_reweight_bin_scales(*d, wl.ENERGY_SCALES, dev(edges)))
    for k, s in enumerate(wl.ENERGY_SCALES):
        ref = oracle.reweight_bin(op, et[1:1 + n], er[1:1 + n], w0[1:1 + n], ch[1:1 + n], s, edges)
        assert_hist_close(got[k], ref, f"scales ragged n={n} s={s}")


def test_scales_fall_back_for_large_binnings(osc):
    n = 20_000
    et, er, w0, ch = wl.events(n, seed=43)
    edges = wl.bin_edges(700, 5.0)                     # three scales of 4 x 700 bins do not fit shared memory
    op = set_params(osc, wl.table1())
    got = host(osc.osc_reweight_bin_scales(dev(et), dev(er), dev(w0), dev(ch), wl.ENERGY_SCALES, dev(edges)))
    for k, s in enumerate(wl.ENERGY_SCALES):
        assert_hist_close(got[k], oracle.reweight_bin(op, et, er, w0, ch, s, edges), f"fallback s={s}")


# ------------------------------------------------------------------------------------------------
# plans: events sorted once, many parameter sets afterwards (osc_plan_*)
# ------------------------------------------------------------------------------------------------
def test_plan_single_sets_vs_oracle_and_k2(osc):
    n = 250_000 + 21
    et, er, w0, ch = wl.events(n, seed=61)
    et[2] = -3.0; ch[3] = 4; er[4] = 1e9
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    plan = osc.osc_plan_create(*d, 1.03, de)
    torch.cuda.synchronize()
    for t in d:                                   # the plan keeps its own sorted copy: scribble over the inputs
        t.zero_()
    d2 = [dev(a) for a in (et, er, w0, ch)]
    for par in (wl.table1(), wl.table1(delta_cp=2.2, hierarchy=-1), wl.table1(rho_g_cm3=0.0, L_km=1300.0, sin2_th23=0.41)):
        op = set_params(osc, par)
        got = host(osc.osc_plan_reweight_bin(plan))
        again = host(osc.osc_plan_reweight_bin(plan))
        assert np.array_equal(got, again)
        assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, 1.03, edges), "plan, single set")
        np.testing.assert_allclose(got, host(osc.osc_reweight_bin(*d2, 1.03, de)), rtol=1e-12, atol=0.0)
    osc.osc_plan_destroy(plan)
    osc.osc_plan_destroy(plan)                    # second destroy of the wrapper is a no-op


@pytest.mark.parametrize("n", [0, 1, 33, 1000])
def test_plan_small_sizes(osc, n):
    et, er, w0, ch = wl.events(max(n, 1), seed=62)
    et, er, w0, ch = et[:n], er[:n], w0[:n], ch[:n]
    edges = wl.bin_edges(7, 4.0)
    op = set_params(osc, wl.table1())
    plan = osc.osc_plan_create(dev(et), dev(er), dev(w0), dev(ch), 0.97, dev(edges))
    assert_hist_close(host(osc.osc_plan_reweight_bin(plan)), oracle.reweight_bin(op, et, er, w0, ch, 0.97, edges),
                      f"plan n={n}")
    pts = [wl.table1(sin2_th23=0.4), wl.table1(sin2_th23=0.6, dm2_32=2.5e-3)]
    got = host(osc.osc_plan_reweight_bin_batch(plan, pts))
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 0.97, edges)
    assert_hist_close(got, ref, f"plan batch n={n}")


def test_plan_batch_grid_and_unrelated_points(osc):
    n = 40_000 + 9
    et, er, w0, ch = wl.events(n, seed=63)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    plan = osc.osc_plan_create(*d, 1.0, dev(edges))
    grid = wl.scan_points()[:64]                       # two dm2_32 groups of 32 points: factorised kernel
    loose = wl.scan_points()[::33][:20]                # unrelated points: one eigen-problem per point
    for name, pts in (("grid", grid), ("loose", loose)):
        got = host(osc.osc_plan_reweight_bin_batch(plan, pts))
        ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
        assert_hist_close(got, ref, f"plan batch {name}")
        direct = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, dev(edges)))
        np.testing.assert_allclose(got, direct, rtol=1e-12, atol=0.0)
        if name == "grid":                             # both main kernels of k4 on the plan's pieces
            for path in K4_PATHS:
                with batch_path(path):
                    forced = host(osc.osc_plan_reweight_bin_batch(plan, pts))
                assert_hist_close(forced, ref, f"plan batch grid, {path}")


def test_outputs_stay_inside_their_buffers(osc):
    """Guard bands around every histogram output (the sanitizer is not available on the GPU pool): each call writes its
    slice of a larger tensor pre-filled with a sentinel, and nothing outside the slice may change."""
    n = 4_000 + 3
    et, er, w0, ch = wl.events(n, seed=71)
    edges = wl.bin_edges(23, 5.0)
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    osc.osc_set_params(**wl.table1())
    grid, loose = wl.scan_points()[:40], wl.scan_points()[::33][:12]
    plan = osc.osc_plan_create(*d, 1.0, de)
    nh = 4 * 23
    calls = [
        (nh, lambda out: osc.osc_reweight_bin(*d, 1.0, de, hist_out=out)),
        (3 * nh, lambda out: osc.osc_reweight_bin_scales(*d, wl.ENERGY_SCALES, de, hist_out=out)),
        (40 * nh, lambda out: osc.osc_reweight_bin_batch(grid, *d, 1.0, de, hist_out=out)),
        (12 * nh, lambda out: osc.osc_reweight_bin_batch(loose, *d, 1.0, de, hist_out=out)),
        (3 * nh, lambda out: osc.osc_reweight_bin_batch(loose[:3], *d, 1.0, de, hist_out=out)),
        (nh, lambda out: osc.osc_plan_reweight_bin(plan, hist_out=out)),
        (40 * nh, lambda out: osc.osc_plan_reweight_bin_batch(plan, grid, hist_out=out)),
        (12 * nh, lambda out: osc.osc_plan_reweight_bin_batch(plan, loose, hist_out=out)),
    ]
    guard = 64
    for k, (size, call) in enumerate(calls):
        buf = torch.full((size + 2 * guard,), -7.0, dtype=torch.float64, device="cuda")
        call(buf[guard:guard + size])
        torch.cuda.synchronize()
        b = host(buf)
        assert np.all(b[:guard] == -7.0) and np.all(b[guard + size:] == -7.0), f"call {k} wrote outside its output"
        assert np.all(b[guard:guard + size] >= 0.0), f"call {k} left part of its output unwritten"
    hist = osc.osc_reweight_bin_batch(loose, *d, 1.0, de)
    buf = torch.full((12 + 2 * guard,), -7.0, dtype=torch.float64, device="cuda")
    osc.osc_neg2lnl(hist, dev(np.ones(nh)), 1.0, out=buf[guard:guard + 12])
    b = host(buf)
    assert np.all(b[:guard] == -7.0) and np.all(b[guard + 12:] == -7.0) and np.all(b[guard:guard + 12] >= 0.0)


# ------------------------------------------------------------------------------------------------
# NEXT-2: Poisson likelihood ratio of the batched histograms on the device (osc_neg2lnl)
# ------------------------------------------------------------------------------------------------
def test_neg2lnl_after_batch(osc):
    pts = wl.scan_points()[::16][:64]
    n = 50_000 + 3
    et, er, w0, ch = wl.events(n, seed=31)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    hist = osc.osc_reweight_bin_batch(pts, *d, 1.0, dev(edges))
    # "data": Poisson draws around the Table-1 expectation (seeded, made on the host from the oracle's histogram)
    ref_hist = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    base = oracle.reweight_bin(oracle.Params(**wl.table1()), et, er, w0, ch, 1.0, edges)
    norm = 0.02
    data = np.random.default_rng(32).poisson(norm * base).astype(np.float64).ravel()
    got = host(osc.osc_neg2lnl(hist, dev(data), norm))
    ref = oracle.neg2lnl(ref_hist, data, norm)
    assert got.shape == (64,)
    scale = float(norm * ref_hist.sum(axis=(1, 2)).max() + data.sum())
    assert np.max(np.abs(got - ref)) <= 1e-12 * scale + 1e-9 * np.max(np.abs(ref))


def test_neg2lnl_edge_cases(osc):
    hist = np.array([[0.0, 2.0, 5.0], [0.0, 2.0, 5.0], [1.0, 0.0, 3.0], [1.0, -1.0, 3.0], [4.0, 4.0, 4.0]])
    data = np.array([0.0, 2.0, 5.0])
    got = host(osc.osc_neg2lnl(dev(hist), dev(data), 1.0))
    ref = oracle.neg2lnl(hist, data, 1.0)
    assert got[0] == 0.0 and got[1] == 0.0
    assert np.isinf(got[2]) and np.isinf(ref[2]) and np.isnan(got[3]) and np.isnan(ref[3])
    assert abs(got[4] - ref[4]) <= 1e-13 * abs(ref[4])
    many = np.random.default_rng(33).uniform(0.0, 30.0, (1000, 37))
    d37 = np.random.default_rng(34).poisson(15.0, 37).astype(np.float64)
    g, r = host(osc.osc_neg2lnl(dev(many), dev(d37), 0.7)), oracle.neg2lnl(many, d37, 0.7)
    np.testing.assert_allclose(g, r, rtol=1e-12)
    assert osc.osc_neg2lnl(dev(many[:0]), dev(d37), 1.0).numel() == 0


# ------------------------------------------------------------------------------------------------
# NEXT-4: bin-centre against event-by-event reweighting over true-energy bins (osc_bin_centre_compare)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,nb", [(0, 5), (1, 1), (777, 13), (300_000, 200)])
def test_bin_centre_compare(osc, n, nb):
    et, _, w0, ch = wl.events(max(n, 1), seed=51)
    et, w0, ch = et[:n].copy(), w0[:n], ch[:n].copy()
    if n > 10:
        et[3] = -1.0; ch[4] = 5; et[5] = 99.0
    edges = wl.bin_edges(nb, 5.0) + 0.05                      # first centre > 0
    op = set_params(osc, wl.table1(delta_cp=1.3, hierarchy=-1))
    he, hc = osc.osc_bin_centre_compare(dev(et), dev(w0), dev(ch), dev(edges))
    re, rc = oracle.bin_centre_compare(op, et, w0, ch, edges)
    assert_hist_close(host(he), re, f"bin-centre compare, event-by-event n={n}")
    assert_hist_close(host(hc), rc, f"bin-centre compare, centre n={n}")


def test_bin_centre_compare_unusable_centre(osc):
    et, _, w0, ch = wl.events(1000, seed=52)
    edges = np.array([-1.0, 1.0, 3.0])                       # first centre is 0: not a usable energy
    op = set_params(osc, wl.table1())
    he, hc = osc.osc_bin_centre_compare(dev(et), dev(w0), dev(ch), dev(edges))
    re, rc = oracle.bin_centre_compare(op, et, w0, ch, edges)
    assert np.all(np.isnan(host(hc)[:, 0])) and np.all(np.isnan(rc[:, 0]))
    assert_hist_close(host(hc)[:, 1], rc[:, 1], "centre, usable bin")
    assert_hist_close(host(he), re, "event-by-event")


def test_bin_centre_compare_768_bins(osc):
    """The largest binning the library accepts: the unit histogram switches to one sub-histogram per warp."""
    n = 60_000 + 1
    et, _, w0, ch = wl.events(n, seed=53)
    edges = wl.bin_edges(768, 5.0) + 0.01
    op = set_params(osc, wl.table1())
    he, hc = osc.osc_bin_centre_compare(dev(et), dev(w0), dev(ch), dev(edges))
    re, rc = oracle.bin_centre_compare(op, et, w0, ch, edges)
    assert_hist_close(host(he), re, "bin-centre compare at 768 bins, event-by-event")
    assert_hist_close(host(hc), rc, "bin-centre compare at 768 bins, centre")


# ------------------------------------------------------------------------------------------------
# multi-GPU host logic with the REAL kernels on one device: every rank of a W-rank job is played in
# turn by this process -- the slices sharding.py hands out (odd offsets, 8-byte-only alignment, ragged ends) go through
# osc_reweight_bin / osc_reweight_bin_batch on device tensors, and the sum (or concatenation) over the ranks is
# compared with the oracle on the whole sample.  The all-reduce itself is covered by tests/test_sharding_gloo.py.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_sharded_reweight_with_the_real_kernels(osc, world):
    from paper_1311_7579_b200 import sharding

    n = 700_000 + 13
    et, er, w0, ch = wl.events(n, seed=81)
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1(delta_cp=0.9))
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    total = np.zeros((4, 50))
    for rank in range(world):
        part = sharding.sharded_reweight_bin(*d, 1.03, de, rank, world, osc.osc_reweight_bin)     # no process group: no reduce
        total += host(part)
        b, e = sharding.shard_bounds(n, rank, world)
        assert_hist_close(host(part), oracle.reweight_bin(op, et[b:e], er[b:e], w0[b:e], ch[b:e], 1.03, edges),
                          f"rank {rank} of {world}")
    assert_hist_close(total, oracle.reweight_bin(op, et, er, w0, ch, 1.03, edges), f"sum over {world} ranks")


@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_sharded_scan_with_the_real_kernels(osc, world):
    from paper_1311_7579_b200 import sharding

    pts = wl.scan_points()[:256]              # 32 dm2_32 groups of 8 points, strided through the list
    n = 20_000 + 3
    et, er, w0, ch = wl.events(n, seed=82)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    ref = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et, er, w0, ch, 1.0, edges)
    owned = sharding.scan_partition(pts, world)
    got = np.full(ref.shape, -1.0)
    for rank in range(world):
        out = host(sharding.sharded_scan(pts, *d, 1.0, de, rank, world, osc.osc_reweight_bin_batch))
        got[owned[rank]] = out[owned[rank]]   # outside a process group a rank fills only its own points
    assert_hist_close(got, ref, f"scan sharded over {world} ranks")


# ------------------------------------------------------------------------------------------------
# asynchrony: parameters are captured at enqueue time; work runs on the caller's stream
# ------------------------------------------------------------------------------------------------
def test_params_captured_at_enqueue_on_side_stream(osc):
    n = 2_000_000
    E = wl.e_true(n, seed=13)
    dE = dev(E)
    pa, pb = wl.table1(), wl.table1(delta_cp=1.0, hierarchy=-1)
    st = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        osc.osc_set_params(**pa)
        out_a = osc.osc_prob(dE, 1, 0, 0, stream=st)
        osc.osc_set_params(**pb)              # must not disturb the launch already enqueued
        out_b = osc.osc_prob(dE, 1, 0, 0, stream=st)
    st.synchronize()
    idx = np.arange(0, n, 997)
    assert_prob_close(host(out_a)[idx], oracle.prob(oracle.Params(**pa), E[idx], 1, 0, 0), "first launch")
    assert_prob_close(host(out_b)[idx], oracle.prob(oracle.Params(**pb), E[idx], 1, 0, 0), "second launch")


def test_host_entry_points(osc):
    n = 50_001
    et, er, w0, ch = wl.events(n, seed=14)
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1())
    assert_prob_close(osc.osc_prob_host(et, 1, 0, 1), oracle.prob(op, et, 1, 0, 1), "osc_prob_host")
    assert_hist_close(osc.osc_reweight_bin_host(et, er, w0, ch, 1.03, edges),
                      oracle.reweight_bin(op, et, er, w0, ch, 1.03, edges), "osc_reweight_bin_host")
    hs = osc.osc_reweight_bin_scales_host(et, er, w0, ch, wl.ENERGY_SCALES, edges)
    assert hs.shape == (3, 4, 50)
    for k, s in enumerate(wl.ENERGY_SCALES):
        assert_hist_close(hs[k], oracle.reweight_bin(op, et, er, w0, ch, s, edges), f"osc_reweight_bin_scales_host {s}")


def test_host_entry_points_in_chunks(osc):
    """Above 2^20 events the host calls send the events in chunks and run the kernel on chunk c while chunk c + 1 is on
    the bus (three chunks here, the last one ragged and odd); the per-chunk histograms are added in chunk order."""
    n = 3_000_001
    et, er, w0, ch = wl.events(n, seed=15)
    et[2_000_000] = float("nan"); ch[1_048_576] = 5; er[1_048_575] = -1.0       # dropped events at the chunk borders
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1(delta_cp=0.7))
    hs = osc.osc_reweight_bin_scales_host(et, er, w0, ch, wl.ENERGY_SCALES, edges)
    again = osc.osc_reweight_bin_scales_host(et, er, w0, ch, wl.ENERGY_SCALES, edges)
    assert np.array_equal(hs, again), "the chunked host call is not bit-reproducible"
    d = [dev(a) for a in (et, er, w0, ch)]
    on_device = host(osc.osc_reweight_bin_scales(*d, wl.ENERGY_SCALES, dev(edges)))
    np.testing.assert_allclose(hs, on_device, rtol=1e-12, atol=0.0)
    assert_hist_close(hs[2], oracle.reweight_bin(op, et, er, w0, ch, wl.ENERGY_SCALES[2], edges), "chunked host call")
    one = osc.osc_reweight_bin_host(et, er, w0, ch, wl.ENERGY_SCALES[0], edges)
    np.testing.assert_allclose(one, hs[0], rtol=1e-12, atol=0.0)


# ------------------------------------------------------------------------------------------------
# BASELINE.json full sizes, in the launch configuration bench.py times.  Every figure BASELINE.md section 4 quotes in
# its parity columns is printed by one of these tests (pytest -s shows them).  The oracle runs on all host cores;
# the whole block costs about two minutes of oracle time on the 16-core GPU box.
# ------------------------------------------------------------------------------------------------
def test_config1_full_size(osc):
    """configs[1] at 1e7 events: run 5 COMPLETE -- all 1e7 x 9 x {nu, nubar} elements against oracle.prob_all -- and the
    other seven runs on 2e5 sampled events (x 9 x 2 = 3.6e6 elements per run) of the same full-size launch.
    (the paper validated all of its 1e7 values, not a sample.)"""
    n = 10_000_000
    E = wl.e_true(n, seed=1)
    dE = dev(E)
    runs = wl.config1_runs()
    out = torch.empty((9, n), dtype=torch.float64, device="cuda")
    idx = np.sort(np.random.Generator(np.random.PCG64(1)).choice(n, 200_000, replace=False))
    idx[:2], idx[-2:] = [0, 1], [n - 2, n - 1]
    d_idx = torch.from_numpy(idx).cuda()
    worst_full = worst_sampled = 0.0
    for r, par in enumerate(runs):
        op = set_params(osc, par)
        for anti in (0, 1):
            osc.osc_prob_all(dE, anti, P_out=out)
            if r == 5:
                worst_full = max(worst_full, assert_prob_close(host(out), oracle.prob_all(op, E, anti),
                                                               f"config1 complete run {r} anti {anti}"))
            else:
                worst_sampled = max(worst_sampled, assert_prob_close(host(out[:, d_idx]), oracle.prob_all(op, E[idx], anti),
                                                                     f"config1 run {r} anti {anti}"))
    print(f"config1 full size: max |dP| = {worst_full:.2e} (run 5, all 1.8e8 elements), "
          f"{worst_sampled:.2e} (7 runs x 3.6e6 sampled elements)")


def test_unitarity_through_nine_independent_calls(osc):
    """osc_prob_all fills five of its nine rows as unitarity complements, so its row and column sums are 1 by
    construction; the nine osc_prob calls assemble every amplitude on its own, and THEIR sums test unitarity."""
    n = 300_000 + 7
    E = wl.e_true(n, seed=15)
    dE = dev(E)
    set_params(osc, wl.config1_runs()[2])
    for anti in (0, 1):
        nine = torch.stack([torch.stack([osc.osc_prob(dE, a, b, anti) for a in range(3)]) for b in range(3)])  # [beta][alpha]
        assert float((nine.sum(0) - 1).abs().max()) < 1e-12 and float((nine.sum(1) - 1).abs().max()) < 1e-12
        alln = osc.osc_prob_all(dE, anti).view(3, 3, n)
        assert float((alln - nine).abs().max()) < 1e-12


def test_config2_full_size(osc):
    """configs[2] at 1e7 events: all three energy scales, k2 (three osc_reweight_bin calls, the step bench.py times) and
    k2s (one osc_reweight_bin_scales call), each histogram DIRECTLY against oracle.reweight_bin on the same 1e7 events;
    bin indices bit-exact on all 1e7 x 3."""
    n = 10_000_000
    et, er, w0, ch = wl.events(n, seed=2)
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1())
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    fused = host(osc.osc_reweight_bin_scales(*d, wl.ENERGY_SCALES, de))
    worst = worst_s = 0.0
    for k, s in enumerate(wl.ENERGY_SCALES):
        ref = oracle.reweight_bin(op, et, er, w0, ch, s, edges)
        worst = max(worst, assert_hist_close(host(osc.osc_reweight_bin(*d, s, de)), ref, f"config2 full, k2, s={s}"))
        worst_s = max(worst_s, assert_hist_close(fused[k], ref, f"config2 full, k2s, s={s}"))
        assert np.array_equal(host(osc.osc_bin_index(d[0], d[1], d[3], s, de)), oracle.bin_index(et, er, ch, s, edges))
    print(f"config2 full size (1e7 events x 3 scales vs the oracle): max rel bin error k2 {worst:.2e}, k2s {worst_s:.2e}; "
          "indices bit-exact")
    # additivity over chunks with odd boundaries (every slice offset and alignment the kernels dispatch on)
    full = host(osc.osc_reweight_bin(*d, 1.03, de))
    cuts = [0, 2_500_001, 5_000_000, 7_499_999, n]
    parts = sum(host(osc.osc_reweight_bin(*[t[a:b] for t in d], 1.03, de)) for a, b in zip(cuts[:-1], cuts[1:]))
    assert np.max(np.abs(parts - full) / np.maximum(full, 1e-300) * (full > 0)) < 1e-12


def test_config2_full_size_plans(osc):
    """The `planned` leg of bench.py (three osc_plan_reweight_bin calls on pre-sorted events) at 1e7 events against
    the oracle's histograms."""
    n = 10_000_000
    et, er, w0, ch = wl.events(n, seed=2)
    edges = wl.bin_edges()
    op = set_params(osc, wl.table1())
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    s = 0.97
    plan = osc.osc_plan_create(*d, s, de)
    got = host(osc.osc_plan_reweight_bin(plan))
    osc.osc_plan_destroy(plan)
    print(f"config2 full size, plan: max rel bin error "
          f"{assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, s, edges), 'config2 full, plan'):.2e}")


def test_config3_full_size(osc):
    """configs[3] by the protocol of SURVEY.md 8(d) (the full 1e6 x 1024 comparison is ~1e9 oracle evaluations, about
    12 minutes on the 16 host cores, so the survey's fallback is what runs): (1) ALL 1024 points on a fixed subsample of
    1e4 events, and (2) the 32 points of the grid diagonal (p = 33 i) on the FULL 1e6 events -- both through the path
    bench.py times (one osc_reweight_bin_batch call, factorised kernel k4); the diagonal also with k5 forced.  The full
    1e6 x 1024 call itself is checked against invariants on every point."""
    pts = wl.scan_points()
    n = 1_000_000
    et, er, w0, ch = wl.events(n, seed=2)
    edges = wl.bin_edges()
    d = [dev(a) for a in (et, er, w0, ch)]
    de = dev(edges)
    # (1) all points, fixed 1e4-event subsample (every 100th event)
    sub = slice(0, n, 100)
    ds = [t[sub].contiguous() for t in d]
    got_sub = host(osc.osc_reweight_bin_batch(pts, *ds, 1.0, de))
    ref_sub = oracle.reweight_bin_batch([oracle.Params(**q) for q in pts], et[sub], er[sub], w0[sub], ch[sub], 1.0, edges)
    e1 = assert_hist_close(got_sub, ref_sub, "config3: 1024 points x 1e4 events (k4)")
    # (2) the full call; its diagonal against the oracle on all 1e6 events
    full = host(osc.osc_reweight_bin_batch(pts, *d, 1.0, de))
    assert full.shape == (1024, 4, 50)
    diag = list(range(0, 1024, 33))
    assert len(diag) == 32
    ref_diag = oracle.reweight_bin_batch([oracle.Params(**pts[p]) for p in diag], et, er, w0, ch, 1.0, edges)
    e2 = assert_hist_close(full[diag], ref_diag, "config3: grid diagonal x 1e6 events (k4, inside the full call)")
    with batch_path("k5"):
        got5 = host(osc.osc_reweight_bin_batch([pts[p] for p in diag], *d, 1.0, de))
    e3 = assert_hist_close(got5, ref_diag, "config3: grid diagonal x 1e6 events (k5)")
    print(f"config3 (SURVEY 8(d) fallback protocol): max rel bin error {e1:.2e} (1024 points x 1e4 events, k4), "
          f"{e2:.2e} (32-point diagonal x 1e6 events, k4), {e3:.2e} (same, k5)")
    # invariants on every point of the full call: P(numu->numu) + P(numu->nue) <= 1, so the channel sums are bounded by
    # the unoscillated histogram of w0; empty cells are the same for every point
    unosc = oracle.reweight_bin(oracle.Params(**wl.table1(L_km=0.0)), et, er, w0, ch, 1.0, edges)   # L = 0: P(mu->mu) = 1
    assert np.all(full >= 0.0) and np.all(np.isfinite(full))
    assert np.all(full[:, 0, :] + full[:, 1, :] <= (unosc[0] + unosc[1]) * (1 + 1e-12))
    assert np.all(full[:, 2, :] + full[:, 3, :] <= (unosc[2] + unosc[3]) * (1 + 1e-12))
    assert np.all((full == 0.0) == (full[0] == 0.0)[None])


@pytest.mark.parametrize("k", range(12))
def test_config4_settings_2e5(osc, k):
    """configs[4]: every (rho, L, hierarchy) setting on 2e5 events, histograms against the oracle."""
    par = wl.sweep_settings()[k]
    n = 200_000 + k
    et, er, w0, ch = wl.events(n, seed=400 + k)
    edges = wl.bin_edges()
    op = set_params(osc, par)
    got = host(osc.osc_reweight_bin(dev(et), dev(er), dev(w0), dev(ch), 1.0, dev(edges)))
    err = assert_hist_close(got, oracle.reweight_bin(op, et, er, w0, ch, 1.0, edges), f"config4 setting {k}")
    print(f"config4 setting {k} (rho {par['rho_g_cm3']}, L {par['L_km']}, h {par['hierarchy']}): max rel bin error {err:.2e}")


def test_config4_1e9_events(osc):
    """configs[4] at its top size: ONE launch over 1e9 device-drawn events (25 GB; the event arrays are 8 GB each, so
    byte offsets beyond 2^32 occur from event 5.4e8 on).
      (a) the launch is bit-reproducible and equals the sum of eight chunk launches to 1e-12;
      (b) two 1e6-event chunks against the oracle: [6e8 + 1, 6e8 + 1e6 + 1) -- odd offset, byte offset 4.8 GB -- and
          [123 456 788, +1e6) -- even offset;
      (c) the high chunk once more INSIDE a 1e9-event launch: with w0 zeroed everywhere else, the full launch must give
          the oracle's histogram of that chunk, so the addressing above 4 GiB meets the oracle directly."""
    free, _ = torch.cuda.mem_get_info()
    if free < 40e9:
        pytest.skip("needs 40 GB of free device memory")
    n = 1_000_000_000
    d = wl.events_device(n, seed=4, device=torch.device("cuda", 0))
    edges = wl.bin_edges()
    de = dev(edges)
    par = wl.table1(rho_g_cm3=5.0, L_km=1300.0, hierarchy=-1)
    op = set_params(osc, par)
    full = host(osc.osc_reweight_bin(*d, 1.0, de))
    assert np.array_equal(full, host(osc.osc_reweight_bin(*d, 1.0, de)))
    m = 125_000_000
    parts = sum(host(osc.osc_reweight_bin(*[t[i:i + m] for t in d], 1.0, de)) for i in range(0, n, m))
    assert np.max(np.abs(parts - full) / np.maximum(full, 1e-300) * (full > 0)) < 1e-12
    worst = 0.0
    for lo in (600_000_001, 123_456_788):
        c = slice(lo, lo + 1_000_000)
        chunk = [host(t[c]) for t in d]
        ref = oracle.reweight_bin(op, *chunk, 1.0, edges)
        worst = max(worst, assert_hist_close(host(osc.osc_reweight_bin(*[t[c] for t in d], 1.0, de)), ref,
                                             f"config4 chunk at {lo} of 1e9"))
        if lo > 600_000_000:
            w_only = torch.zeros_like(d[2])
            w_only[c] = d[2][c]
            inside = host(osc.osc_reweight_bin(d[0], d[1], w_only, d[3], 1.0, de))
            del w_only
            worst = max(worst, assert_hist_close(inside, ref, "config4: chunk above 4 GiB inside the 1e9-event launch"))
    print(f"config4 at 1e9 events: chunk sums equal the full launch to 1e-12; chunks vs oracle max rel bin error {worst:.2e}")


def test_paper_validation_replay(osc):
    """1e7 energies uniform in 0-30 GeV, residuals ~1e-12 in fp64 (A12: floored at 1e-3 GeV)."""
    n = 10_000_000
    E = wl.validation_energies(n, seed=4)
    op = set_params(osc, wl.table1())
    dE = dev(E)
    idx = np.random.Generator(np.random.PCG64(4)).choice(n, 40_000, replace=False)
    idx[:64] = np.argsort(E)[:64]          # the lowest energies = the largest phases
    for fin, fout, anti in ((1, 1, 0), (1, 0, 0), (1, 0, 1)):
        got = host(osc.osc_prob(dE, fin, fout, anti))
        err = assert_prob_close(got[idx], oracle.prob(op, E[idx], fin, fout, anti), "validation replay")
        print(f"validation replay {fin}->{fout} anti={anti}: max |dP| = {err:.2e}")
