"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md "Input recipe").

This module holds NO arithmetic of the method (no mixing matrix, no probability, no binning):
it only draws the arrays that both the CUDA path and the test oracle are handed, byte-identical.
It imports neither the CUDA binding nor ``oracle``.

The arrays stand in for the paper's workloads -- a Landau-sampled toy beam spectrum with unstated
parameters, the U(0,30) GeV validation set and T2K Monte Carlo
(PAPER.md:162), none of which is available -- with the shapes and distributions that
BASELINE.json:configs fixes.
"""
from __future__ import annotations

import math
from typing import Dict, List, Tuple

import numpy as np

# Table 1 of the paper, normal hierarchy.  "dm2_12" printed there is
# read as dm2_21 (reading A4).
TABLE1: Dict[str, float] = dict(sin2_th12=0.311, sin2_th23=0.5, sin2_th13=0.0251, dm2_32=2.4e-3,
                                dm2_21=7.6e-5, delta_cp=0.0, rho_g_cm3=2.6, L_km=295.0, hierarchy=1)

PARAM_FIELDS = ("sin2_th12", "sin2_th23", "sin2_th13", "dm2_32", "dm2_21", "delta_cp", "rho_g_cm3",
                "L_km", "hierarchy")

N_CHANNELS = 4      # numu->numu, numu->nue, numubar->numubar, numubar->nuebar (configs[2])
N_BINS = 50         # configs[2]: 50 bins over 0-5 GeV
E_LO, E_HI = 0.1, 10.0
ENERGY_SCALES = (0.97, 1.00, 1.03)


def table1(**overrides) -> Dict[str, float]:
    d = dict(TABLE1)
    d.update(overrides)
    return d


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def e_true(n: int, seed: int = 0) -> np.ndarray:
    """E_true = clamp(exp(ln 0.7 + 0.5 z), 0.1, 10) GeV, z ~ N(0,1)  (configs[0])."""
    z = _rng(seed).standard_normal(n)
    return np.clip(np.exp(math.log(0.7) + 0.5 * z), E_LO, E_HI)


def events(n: int, seed: int = 2) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
    """(E_true, E_reco, w0, channel) with the configs[2] layout.

    E_true as in ``e_true``; E_reco = E_true (1 + 0.1 z'); w0 ~ U[0.5, 1.5); channel ~ U{0..3} int8.
    """
    rng = _rng(seed)
    z = rng.standard_normal(n)
    et = np.clip(np.exp(math.log(0.7) + 0.5 * z), E_LO, E_HI)
    er = et * (1.0 + 0.1 * rng.standard_normal(n))
    w0 = rng.uniform(0.5, 1.5, n)
    ch = rng.integers(0, N_CHANNELS, n, dtype=np.int8)
    return et, er, w0, ch


def bin_edges(n_bins: int = N_BINS, hi: float = 5.0) -> np.ndarray:
    """edges[i] = hi * i / n_bins in fp64, i = 0..n_bins  (configs[2]: 50 bins over 0-5 GeV)."""
    return np.array([hi * i / float(n_bins) for i in range(n_bins + 1)], dtype=np.float64)


def config1_runs(seed: int = 1, n_delta: int = 4) -> List[Dict[str, float]]:
    """configs[1]: delta_cp ~ U[-pi, pi) per run (n_delta seeded draws) x both hierarchies."""
    deltas = _rng(seed).uniform(-math.pi, math.pi, n_delta)
    return [table1(delta_cp=float(d), hierarchy=h) for d in deltas for h in (1, -1)]


def scan_points(seed: int = 3, n_side: int = 32) -> List[Dict[str, float]]:
    """configs[3]: n_side x n_side inclusive grid, sin2_th23 in [0.3, 0.7] x dm2_32 in [2.0e-3, 3.0e-3],
    delta_cp ~ U[-pi, pi) per point; point p = n_side * i_th23 + j_dm2; normal hierarchy."""
    deltas = _rng(seed).uniform(-math.pi, math.pi, n_side * n_side)
    pts = []
    for i in range(n_side):
        for j in range(n_side):
            s23 = 0.3 + 0.4 * i / (n_side - 1)
            dm = (2.0 + 1.0 * j / (n_side - 1)) * 1e-3
            pts.append(table1(sin2_th23=s23, dm2_32=dm, delta_cp=float(deltas[n_side * i + j])))
    return pts


def sweep_settings() -> List[Dict[str, float]]:
    """configs[4]: rho in {0, 2.6, 5.0} x L in {295, 1300} x both hierarchies."""
    return [table1(rho_g_cm3=rho, L_km=L, hierarchy=h)
            for rho in (0.0, 2.6, 5.0) for L in (295.0, 1300.0) for h in (1, -1)]


def validation_energies(n: int, seed: int = 4, floor: float = 1e-3) -> np.ndarray:
    """The paper's validation draw: uniform in (0, 30] GeV, floored at 1e-3 GeV (A12)."""
    return np.maximum(_rng(seed).uniform(0.0, 30.0, n), floor)


def events_device(n: int, seed: int, device):
    """configs[4] at sizes that do not fit a host array (up to 1e9 events = 25 GB): the same laws as
    ``events`` drawn with torch's device generator.  Returns torch tensors on ``device``."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    et = torch.empty(n, dtype=torch.float64, device=device)
    et.normal_(0.0, 1.0, generator=g).mul_(0.5).add_(math.log(0.7)).exp_().clamp_(E_LO, E_HI)
    er = torch.empty(n, dtype=torch.float64, device=device)
    er.normal_(0.0, 1.0, generator=g).mul_(0.1).add_(1.0).mul_(et)
    w0 = torch.empty(n, dtype=torch.float64, device=device)
    w0.uniform_(0.5, 1.5, generator=g)
    ch = torch.randint(0, N_CHANNELS, (n,), dtype=torch.int8, device=device, generator=g)
    return et, er, w0, ch
