"""Pins for the CPU oracle.  CPU only.

Each test checks ``oracle/`` against something that is NOT the oracle: a closed form, a symmetry,
brute force, or a value the paper prints.  The formulas live in tests/physics_ref.py and are built
by different routes than the oracle's (see that file's header).
"""
from __future__ import annotations

import itertools
import math
import os

import numpy as np
import pytest

import oracle
import physics_ref as ref
from paper_1311_7579_b200 import workloads

FLAVOURS = (0, 1, 2)


def _random_params(rng, rho=None, L=None, hierarchy=None, delta=None):
    return oracle.Params(
        sin2_th12=rng.uniform(0.2, 0.4), sin2_th23=rng.uniform(0.3, 0.7), sin2_th13=rng.uniform(0.01, 0.05),
        dm2_32=rng.uniform(2.0e-3, 3.0e-3), dm2_21=rng.uniform(6e-5, 9e-5),
        delta_cp=rng.uniform(-math.pi, math.pi) if delta is None else delta,
        rho_g_cm3=rng.uniform(0.0, 6.0) if rho is None else rho,
        L_km=rng.uniform(100.0, 1500.0) if L is None else L,
        hierarchy=int(rng.choice([-1, 1])) if hierarchy is None else hierarchy)


def _U_m2(p: oracle.Params):
    return (ref.pmns(p.sin2_th12, p.sin2_th23, p.sin2_th13, p.delta_cp),
            ref.masses(p.dm2_32, p.dm2_21, p.hierarchy))


# ---------------------------------------------------------------------------------------------------
# constants: the oracle's typed-in K_PHASE / K_MATTER / Y_E against values derived from CODATA
# ---------------------------------------------------------------------------------------------------
def test_constants_match_codata_derivation():
    assert ref.K_PHASE == pytest.approx(2.5338653580781979, rel=1e-14)
    assert ref.K_MATTER == pytest.approx(1.5264932449499478e-4, rel=1e-14)


# ---------------------------------------------------------------------------------------------------
# P1  rho = 0  ==  vacuum mass-state sum (eq. 1.1 as read in A1), all 9 transitions, nu and nubar
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(6))
def test_p1_vacuum_formula(seed):
    rng = np.random.default_rng(100 + seed)
    p = _random_params(rng, rho=0.0)
    U, m2 = _U_m2(p)
    E = rng.uniform(0.1, 10.0, 7)
    for antinu in (0, 1):
        got = oracle.prob_all(p, E, antinu)
        for a, b in itertools.product(FLAVOURS, FLAVOURS):
            want = [ref.vacuum_prob(U, m2, p.L_km, e, a, b, bool(antinu)) for e in E]
            assert np.max(np.abs(got[3 * b + a] - want)) < 2e-13, (a, b, antinu)
            single = oracle.prob(p, E, a, b, antinu)
            assert np.array_equal(single, got[3 * b + a])


# ---------------------------------------------------------------------------------------------------
# P2  unitarity
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
def test_p2_unitarity(seed):
    rng = np.random.default_rng(200 + seed)
    p = _random_params(rng)
    E = rng.uniform(0.1, 10.0, 64)
    for antinu in (0, 1):
        P = oracle.prob_all(p, E, antinu).reshape(3, 3, -1)   # [beta, alpha, event]
        assert np.max(np.abs(P.sum(axis=0) - 1.0)) < 1e-13
        assert np.max(np.abs(P.sum(axis=1) - 1.0)) < 1e-13
        S = oracle.evolution(p, float(E[0]), antinu)
        assert np.max(np.abs(S.conj().T @ S - np.eye(3))) < 1e-15


# ---------------------------------------------------------------------------------------------------
# P3  theta13 = 0, dm2_21 = 0: two-flavour formula, independent of rho (exactly degenerate eigenvalues)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rho", [0.0, 2.6, 50.0])
@pytest.mark.parametrize("hierarchy", [1, -1])
def test_p3_two_flavour(rho, hierarchy):
    s2_23 = 0.42
    p = oracle.Params(0.311, s2_23, 0.0, 2.4e-3, 0.0, 0.7, rho, 295.0, hierarchy)
    E = np.array([0.1, 0.3, 0.6, 1.0, 2.5, 10.0])
    sin2_2t = 4.0 * s2_23 * (1.0 - s2_23)
    dm31 = hierarchy * 2.4e-3
    for antinu in (0, 1):
        want = [ref.two_flavour_survival(sin2_2t, dm31, 295.0, e) for e in E]
        assert np.max(np.abs(oracle.prob(p, E, 1, 1, antinu) - want)) < 1e-13
        assert np.max(np.abs(oracle.prob(p, E, 0, 0, antinu) - 1.0)) < 1e-13
        assert np.max(np.abs(oracle.prob(p, E, 1, 0, antinu))) < 1e-13
        assert np.max(np.abs(oracle.prob(p, E, 1, 2, antinu) - (1.0 - np.array(want)))) < 1e-13


# ---------------------------------------------------------------------------------------------------
# P4  delta = 0  =>  P(a->b) = P(b->a), in vacuum and in constant-density matter
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rho", [0.0, 2.6])
def test_p4_t_symmetry(rho):
    rng = np.random.default_rng(400)
    p = _random_params(rng, rho=rho, delta=0.0)
    E = rng.uniform(0.1, 10.0, 32)
    for antinu in (0, 1):
        P = oracle.prob_all(p, E, antinu).reshape(3, 3, -1)
        assert np.max(np.abs(P - P.transpose(1, 0, 2))) < 1e-14
    # and T is violated when delta != 0 (the test would be vacuous if P were always symmetric)
    q = _random_params(rng, rho=rho, delta=1.1)
    Pq = oracle.prob_all(q, E, 0).reshape(3, 3, -1)
    assert np.max(np.abs(Pq - Pq.transpose(1, 0, 2))) > 1e-3


# ---------------------------------------------------------------------------------------------------
# P5  L = 0  =>  P = identity
# ---------------------------------------------------------------------------------------------------
def test_p5_zero_baseline():
    rng = np.random.default_rng(500)
    p = _random_params(rng, L=0.0)
    E = rng.uniform(0.1, 10.0, 16)
    for antinu in (0, 1):
        P = oracle.prob_all(p, E, antinu).reshape(3, 3, -1)
        assert np.max(np.abs(P - np.eye(3)[:, :, None])) < 1e-15


# ---------------------------------------------------------------------------------------------------
# P6  brute force: RK4 integration of i dpsi/dl = (K/E) H psi on tiny event sets
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", [
    dict(),                                                # Table 1, normal
    dict(hierarchy=-1, delta_cp=-1.2),
    dict(rho_g_cm3=5.0, L_km=1300.0, delta_cp=2.0),
])
def test_p6_rk4_schroedinger(case):
    p = oracle.Params(**workloads.table1(**case))
    U, m2 = _U_m2(p)
    for E in (0.35, 0.6, 2.0):
        for antinu in (0, 1):
            H = ref.hamiltonian(U, m2, p.rho_g_cm3, E, bool(antinu))
            want = ref.rk4_probs(H, p.L_km, E, n_steps=12000)
            got = oracle.prob_all(p, [E], antinu).reshape(3, 3)
            assert np.max(np.abs(got - want)) < 2e-11, (case, E, antinu)


def test_eigenvalues_against_lapack():
    rng = np.random.default_rng(650)
    for _ in range(20):
        p = _random_params(rng)
        U, m2 = _U_m2(p)
        E = float(rng.uniform(0.1, 10.0))
        for antinu in (0, 1):
            H = ref.hamiltonian(U, m2, p.rho_g_cm3, E, bool(antinu))
            want = np.linalg.eigvalsh(H)
            got = oracle.eigenvalues(p, E, antinu)
            assert np.max(np.abs(got - want)) < 1e-17 + 1e-13 * np.max(np.abs(want))


# ---------------------------------------------------------------------------------------------------
# P7  one-mass-scale MSW closed form (dm2_21 = 0): pins K_MATTER, Y_E and the antineutrino sign
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rho", [2.6, 50.0])
@pytest.mark.parametrize("hierarchy", [1, -1])
def test_p7_msw_one_mass_scale(rho, hierarchy):
    s2_13, s2_23 = 0.0251, 0.55
    p = oracle.Params(0.311, s2_23, s2_13, 2.4e-3, 0.0, 0.3, rho, 1300.0, hierarchy)
    th13 = math.asin(math.sqrt(s2_13))
    dm31 = hierarchy * 2.4e-3
    E = np.array([0.5, 1.0, 2.0, 4.0, 8.0])
    for antinu in (0, 1):
        trans = np.array([ref.msw_two_flavour(th13, dm31, ref.matter_term(rho, e, bool(antinu)), 1300.0, e)
                          for e in E])
        assert np.max(np.abs(oracle.prob(p, E, 0, 0, antinu) - (1.0 - trans))) < 1e-13
        assert np.max(np.abs(oracle.prob(p, E, 1, 0, antinu) - s2_23 * trans)) < 1e-13
        assert np.max(np.abs(oracle.prob(p, E, 0, 2, antinu) - (1.0 - s2_23) * trans)) < 1e-13
    # matter enhances nu and suppresses nubar for the normal hierarchy, reversed for the inverted one
    e = np.array([3.0])
    nu, nubar = oracle.prob(p, e, 1, 0, 0)[0], oracle.prob(p, e, 1, 0, 1)[0]
    assert (nu > nubar) == (hierarchy == 1)


# ---------------------------------------------------------------------------------------------------
# P8  theta13 = 0: nu_e survival is a two-level (theta12, dm2_21) MSW problem
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rho", [0.0, 2.6, 10.0])
def test_p8_solar_sector(rho):
    s2_12 = 0.311
    p = oracle.Params(s2_12, 0.5, 0.0, 2.4e-3, 7.6e-5, 1.0, rho, 1300.0, 1)
    th12 = math.asin(math.sqrt(s2_12))
    E = np.array([0.1, 0.2, 0.5, 1.0, 3.0])
    for antinu in (0, 1):
        trans = np.array([ref.msw_two_flavour(th12, 7.6e-5, ref.matter_term(rho, e, bool(antinu)), 1300.0, e)
                          for e in E])
        assert np.max(np.abs(oracle.prob(p, E, 0, 0, antinu) - (1.0 - trans))) < 1e-13


# ---------------------------------------------------------------------------------------------------
# P9  P(nu_e -> nu_e) does not depend on theta23 or delta
# ---------------------------------------------------------------------------------------------------
def test_p9_pee_independent_of_th23_delta():
    E = np.linspace(0.1, 10.0, 40)
    base = oracle.prob(oracle.Params(**workloads.table1()), E, 0, 0, 0)
    for s23, d in ((0.3, 0.0), (0.7, 1.0), (0.45, -2.5)):
        other = oracle.prob(oracle.Params(**workloads.table1(sin2_th23=s23, delta_cp=d)), E, 0, 0, 0)
        assert np.max(np.abs(other - base)) < 1e-14


# ---------------------------------------------------------------------------------------------------
# P10  CP / CPT relations and the sign convention of delta (A6)
# ---------------------------------------------------------------------------------------------------
def test_p10_cpt_and_delta_sign():
    rng = np.random.default_rng(1000)
    p = _random_params(rng, rho=0.0)
    E = rng.uniform(0.1, 10.0, 16)
    Pn = oracle.prob_all(p, E, 0).reshape(3, 3, -1)
    Pa = oracle.prob_all(p, E, 1).reshape(3, 3, -1)
    assert np.max(np.abs(Pa - Pn.transpose(1, 0, 2))) < 1e-14          # vacuum: Pbar(a->b) = P(b->a)
    # antineutrinos in matter == neutrinos with delta -> -delta and the opposite matter sign, which a
    # vanishing density makes testable without a "negative rho": compare at rho = 0 only for delta.
    q = oracle.Params(p.sin2_th12, p.sin2_th23, p.sin2_th13, p.dm2_32, p.dm2_21, -p.delta_cp, 0.0, p.L_km,
                      p.hierarchy)
    assert np.max(np.abs(oracle.prob_all(q, E, 0) - oracle.prob_all(p, E, 1))) < 1e-14
    # delta = -pi/2 enhances nu_mu -> nu_e for neutrinos and suppresses it for antineutrinos (A6)
    e = np.array([0.6])
    lo = oracle.Params(**workloads.table1(delta_cp=-math.pi / 2, rho_g_cm3=0.0))
    hi = oracle.Params(**workloads.table1(delta_cp=+math.pi / 2, rho_g_cm3=0.0))
    assert oracle.prob(lo, e, 1, 0, 0)[0] > oracle.prob(hi, e, 1, 0, 0)[0]
    assert oracle.prob(lo, e, 1, 0, 1)[0] < oracle.prob(hi, e, 1, 0, 1)[0]


# ---------------------------------------------------------------------------------------------------
# paper-printed value: the trough of P(numu->numu) "at 0.6 GeV", figure precision
# ---------------------------------------------------------------------------------------------------
def _golden(name):
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            vals[k] = float(v)
    return vals


def test_paper_fig1_trough(table1_params):
    g = _golden("paper_fig1_trough.txt")
    E = np.linspace(0.3, 1.5, 2401)
    P = oracle.prob(table1_params, E, 1, 1, 0)
    e_min = E[int(np.argmin(P))]
    assert g["lo"] <= e_min <= g["hi"]
    assert oracle.prob(table1_params, [g["trough_E_GeV"]], 1, 1, 0)[0] < g["p_max"]


# ---------------------------------------------------------------------------------------------------
# A11: unusable energies give NaN
# ---------------------------------------------------------------------------------------------------
def test_bad_energies_are_nan(table1_params):
    P = oracle.prob(table1_params, [0.0, -1.0, float("nan"), float("inf"), 0.6], 1, 1, 0)
    assert np.all(np.isnan(P[:4])) and np.isfinite(P[4])


# ---------------------------------------------------------------------------------------------------
# P11  histogram: brute force, L = 0, edge placement, permutation invariance, drop rule
# ---------------------------------------------------------------------------------------------------
def _brute_hist(E_reco, w, ch, s, edges, n_ch=4):
    nb = len(edges) - 1
    H = [[0.0] * nb for _ in range(n_ch)]
    for j in range(len(w)):
        x = np.float64(s) * np.float64(E_reco[j])
        for i in range(nb):
            if edges[i] <= x < edges[i + 1]:
                H[int(ch[j])][i] += float(w[j])
                break
    return np.array(H)


def test_p11_zero_baseline_is_plain_weighted_histogram():
    et, er, w0, ch = workloads.events(1000, seed=11)
    edges = workloads.bin_edges()
    p = oracle.Params(**workloads.table1(L_km=0.0))
    # L = 0: P(mu->mu) = 1 (channels 0, 2), P(mu->e) = 0 (channels 1, 3)
    w = np.where(ch % 2 == 0, w0, 0.0)
    for s in workloads.ENERGY_SCALES:
        got = oracle.reweight_bin(p, et, er, w0, ch, s, edges)
        want = _brute_hist(er, w, ch, s, edges)
        assert np.max(np.abs(got - want)) < 1e-12


def test_p11_brute_force_with_oscillation(table1_params):
    et, er, w0, ch = workloads.events(600, seed=12)
    edges = workloads.bin_edges()
    P = np.empty(600)
    table = [(1, 1, 0), (1, 0, 0), (1, 1, 1), (1, 0, 1)]
    for c, (a, b, anti) in enumerate(table):
        m = ch == c
        P[m] = oracle.prob(table1_params, et[m], a, b, anti)
    got = oracle.reweight_bin(table1_params, et, er, w0, ch, 1.03, edges)
    want = _brute_hist(er, w0 * P, ch, 1.03, edges)
    assert np.max(np.abs(got - want) / np.maximum(want, 1e-300)) < 1e-12
    # bin indices: same rule, integer exact
    idx = oracle.bin_index(et, er, ch, 1.03, edges)
    x = np.float64(1.03) * er
    want_idx = np.searchsorted(edges, x, side="right") - 1
    want_idx[(x < edges[0]) | (x >= edges[-1])] = -1
    assert np.array_equal(idx, want_idx.astype(np.int32))


def test_p11_edges_upper_bin_and_drop_rule(table1_params):
    edges = workloads.bin_edges()
    er = np.array([edges[0], edges[1], edges[7], edges[49], edges[50], -0.1, np.nextafter(edges[50], 0.0),
                   float("nan"), 1.0, 1.0, 1.0])
    et = np.full(er.size, 0.8)
    et[8] = 0.0          # unusable true energy -> dropped
    ch = np.zeros(er.size, dtype=np.int8)
    ch[9] = 4            # channel out of range -> dropped
    ch[10] = -1
    idx = oracle.bin_index(et, er, ch, 1.0, edges)
    assert idx.tolist() == [0, 1, 7, 49, -1, -1, 49, -1, -1, -1, -1]
    w0 = np.ones(er.size)
    H = oracle.reweight_bin(table1_params, et, er, w0, ch, 1.0, edges)
    pmm = oracle.prob(table1_params, [0.8], 1, 1, 0)[0]
    assert H[0, 49] == pytest.approx(2 * pmm, rel=1e-15)
    assert H.sum() == pytest.approx(5 * pmm, rel=1e-14)
    assert np.all(H[1:] == 0.0)


def test_p11_sum_and_permutation_invariance(table1_params):
    et, er, w0, ch = workloads.events(4000, seed=13)
    edges = workloads.bin_edges()
    H = oracle.reweight_bin(table1_params, et, er, w0, ch, 1.0, edges)
    perm = np.random.default_rng(0).permutation(et.size)
    Hp = oracle.reweight_bin(table1_params, et[perm], er[perm], w0[perm], ch[perm], 1.0, edges)
    assert np.max(np.abs(H - Hp) / np.maximum(H, 1e-300)) < 1e-15
    idx = oracle.bin_index(et, er, ch, 1.0, edges)
    table = [(1, 1, 0), (1, 0, 0), (1, 1, 1), (1, 0, 1)]
    total = 0.0
    for c, (a, b, anti) in enumerate(table):
        m = (ch == c) & (idx >= 0)
        total += float(np.sum(w0[m] * oracle.prob(table1_params, et[m], a, b, anti)))
    assert H.sum() == pytest.approx(total, rel=1e-13)


# ---------------------------------------------------------------------------------------------------
# P12  batched slice == single call; energy scales share the weights
# ---------------------------------------------------------------------------------------------------
def test_p12_batch_slices_and_energy_scales():
    et, er, w0, ch = workloads.events(300, seed=14)
    edges = workloads.bin_edges()
    pts = [oracle.Params(**d) for d in workloads.scan_points(seed=3, n_side=3)]
    B = oracle.reweight_bin_batch(pts, et, er, w0, ch, 1.0, edges)
    assert B.shape == (9, 4, 50)
    for k, q in enumerate(pts):
        assert np.array_equal(B[k], oracle.reweight_bin(q, et, er, w0, ch, 1.0, edges))
    one_bin = np.array([-1e30, 1e30])
    totals = [oracle.reweight_bin(pts[4], et, er, w0, ch, s, one_bin) for s in workloads.ENERGY_SCALES]
    assert np.array_equal(totals[0], totals[1]) and np.array_equal(totals[1], totals[2])


# ------------------------------------------------------------------------------------------------
# P13: binned Poisson likelihood ratio (eq. 2.1; reading R5)
# ------------------------------------------------------------------------------------------------
def test_p13_neg2lnl_against_scipy_poisson_pmf():
    """For integer data -2 ln lambda = -2 [ln Pois(D | mu) - ln Pois(D | D)], bin by bin (scipy's pmf, not a
    retyped formula)."""
    from scipy.stats import poisson

    rng = np.random.default_rng(5)
    mu = rng.uniform(0.05, 400.0, (7, 60))
    D = rng.poisson(mu[3]).astype(np.float64)
    D[::11] = 0.0
    got = oracle.neg2lnl(mu, D, 1.0)
    for p in range(mu.shape[0]):
        sat = np.where(D > 0, poisson.logpmf(D, np.maximum(D, 1e-300)), 0.0)
        ref = -2.0 * np.sum(poisson.logpmf(D, mu[p]) - sat)
        assert abs(got[p] - ref) <= 1e-9 * max(abs(ref), 1.0)


def test_p13_neg2lnl_closed_forms():
    rng = np.random.default_rng(6)
    mu = rng.uniform(0.1, 50.0, (3, 40))
    # data equal to the expectation: exactly the saturated model
    assert np.all(np.abs(oracle.neg2lnl(mu[1:2], mu[1], 1.0)) < 1e-12)
    # empty data: 2 * sum(mu); the normalisation multiplies the expectation
    z = np.zeros(40)
    np.testing.assert_allclose(oracle.neg2lnl(mu, z, 1.0), 2.0 * mu.sum(axis=1), rtol=1e-14)
    np.testing.assert_allclose(oracle.neg2lnl(mu, z, 2.5), 5.0 * mu.sum(axis=1), rtol=1e-14)
    # one bin, D = e * mu: 2 [mu - e mu + e mu] = 2 mu
    got = oracle.neg2lnl(np.array([[3.0]]), np.array([3.0 * math.e]), 1.0)
    assert abs(got[0] - 6.0) < 1e-13
    # scaling norm and 1/hist together changes nothing; the result is >= 0 and additive over bins
    D = rng.poisson(mu[0]).astype(np.float64)
    a = oracle.neg2lnl(mu, D, 1.0)
    np.testing.assert_allclose(oracle.neg2lnl(mu / 4.0, D, 4.0), a, rtol=1e-13)
    assert np.all(a >= 0.0)
    np.testing.assert_allclose(oracle.neg2lnl(mu[:, :17], D[:17], 1.0) + oracle.neg2lnl(mu[:, 17:], D[17:], 1.0), a,
                               rtol=1e-13)
    # degenerate bins: mu = 0 with and without data; invalid entries
    assert oracle.neg2lnl(np.array([[0.0, 1.0]]), np.array([0.0, 1.0]), 1.0)[0] == 0.0
    assert np.isinf(oracle.neg2lnl(np.array([[0.0, 1.0]]), np.array([2.0, 1.0]), 1.0)[0])
    assert np.isnan(oracle.neg2lnl(np.array([[-1.0, 1.0]]), np.array([2.0, 1.0]), 1.0)[0])


# ------------------------------------------------------------------------------------------------
# P14: bin-centre against event-by-event reweighting over true-energy bins
# ------------------------------------------------------------------------------------------------
def test_p14_bin_centre_compare_against_numpy_histograms():
    rng = np.random.default_rng(8)
    n = 4000
    E = rng.uniform(0.2, 3.0, n)
    w0 = rng.uniform(0.5, 1.5, n)
    ch = rng.integers(0, 4, n).astype(np.int8)
    edges = np.linspace(0.25, 2.75, 11)
    p = oracle.Params(**workloads.table1(delta_cp=0.7))
    he, hc = oracle.bin_centre_compare(p, E, w0, ch, edges)
    chan = [(1, 1, 0), (1, 0, 0), (1, 1, 1), (1, 0, 1)]
    centres = 0.5 * (edges[:-1] + edges[1:])
    for c, (fi, fo, an) in enumerate(chan):
        m = ch == c
        ev, _ = np.histogram(E[m], bins=edges, weights=w0[m] * oracle.prob(p, E[m], fi, fo, an))
        un, _ = np.histogram(E[m], bins=edges, weights=w0[m])
        # numpy's last bin is closed on the right; no event sits on that edge here
        np.testing.assert_allclose(he[c], ev, rtol=1e-12)
        np.testing.assert_allclose(hc[c], un * oracle.prob(p, centres, fi, fo, an), rtol=1e-12)


def test_p14_bin_centre_limits():
    rng = np.random.default_rng(9)
    edges = np.linspace(0.5, 1.5, 6)
    centres = 0.5 * (edges[:-1] + edges[1:])
    w0 = rng.uniform(0.5, 1.5, 500)
    ch = rng.integers(0, 4, 500).astype(np.int8)
    # every event exactly at a bin centre: the two methods are the same calculation
    E = centres[rng.integers(0, 5, 500)]
    p = oracle.Params(**workloads.table1())
    he, hc = oracle.bin_centre_compare(p, E, w0, ch, edges)
    np.testing.assert_allclose(hc, he, rtol=1e-13)
    # L = 0: P = delta, both methods give the unoscillated histogram (survival) or zero (appearance)
    p0 = oracle.Params(**workloads.table1(L_km=0.0))
    E = rng.uniform(0.5, 1.5, 500)
    he, hc = oracle.bin_centre_compare(p0, E, w0, ch, edges)
    np.testing.assert_allclose(hc, he, rtol=1e-13, atol=1e-30)
    assert np.all(np.abs(he[[1, 3]]) < 1e-30)
    # the effect the paper describes: a 25 MeV bin next to the oscillation maximum, flat spectrum inside the bin
    E = np.linspace(0.6, 0.625, 2001)[:-1] + 0.0125 / 2000
    he, hc = oracle.bin_centre_compare(p, E, np.ones_like(E), np.zeros(E.size, np.int8), np.array([0.6, 0.625]))
    # near the minimum of P(numu -> numu) the curvature makes the bin-centre value too LOW by a few per cent
    assert -0.06 < hc[0, 0] / he[0, 0] - 1.0 < -0.005
