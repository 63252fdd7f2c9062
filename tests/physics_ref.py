"""Independent textbook formulas used ONLY to pin the oracle (tests/test_oracle_pins.py).

Nothing here is shared with ``oracle/`` or with the CUDA path:
  * the unit-conversion constants are re-derived from CODATA/PDG values instead of being typed in;
  * the PMNS matrix is built as the matrix product R23 . U13(delta) . R12 instead of entry by entry;
  * probabilities come from closed forms (vacuum mass-state sum, two-flavour formula, one-mass-scale
    MSW formula) or from brute-force RK4 integration of the Schroedinger equation, never from an
    eigen-decomposition of the 3x3 matter Hamiltonian.
"""
from __future__ import annotations

import math

import numpy as np

# CODATA 2018 exact SI values and PDG G_F.
_H_PLANCK = 6.62607015e-34          # J s (exact)
_C_LIGHT = 299792458.0              # m / s (exact)
_E_CHARGE = 1.602176634e-19         # C (exact)
HBARC_EV_M = _H_PLANCK * _C_LIGHT / (2.0 * math.pi * _E_CHARGE)   # hbar c in eV m = 1.97326980459...e-7
G_F_GEV2 = 1.1663787e-5             # Fermi constant / (hbar c)^3, GeV^-2
N_A = 6.02214076e23                 # Avogadro, 1/mol (nucleons per gram)
Y_E = 0.5                           # electrons per nucleon (reading A3)

# phase = m^2 L / (2 E hbar c):  m^2 [eV^2] * L[km]*1e3 m / (2 * E[GeV]*1e9 eV * hbarc [eV m])
K_PHASE = 1.0e3 / (2.0 * 1.0e9 * HBARC_EV_M)
# A = 2 sqrt2 G_F N_e E, N_e = Y_e rho N_A per cm^3; (hbar c)^3 in GeV^3 cm^3; result eV^2 per (GeV g/cm^3)
_HBARC_GEV_CM = HBARC_EV_M * 1e-9 * 1e2
K_MATTER = 2.0 * math.sqrt(2.0) * G_F_GEV2 * (_HBARC_GEV_CM ** 3) * N_A * 1e9 * 1e9


def pmns(s2_12: float, s2_23: float, s2_13: float, delta: float) -> np.ndarray:
    """U = R23 . U13(delta) . R12, rows = flavours (e, mu, tau), columns = mass states."""
    t12, t23, t13 = (math.asin(math.sqrt(v)) for v in (s2_12, s2_23, s2_13))
    c12, s12, c23, s23, c13, s13 = (math.cos(t12), math.sin(t12), math.cos(t23), math.sin(t23),
                                    math.cos(t13), math.sin(t13))
    r23 = np.array([[1, 0, 0], [0, c23, s23], [0, -s23, c23]], dtype=complex)
    u13 = np.array([[c13, 0, s13 * np.exp(-1j * delta)], [0, 1, 0], [-s13 * np.exp(1j * delta), 0, c13]],
                   dtype=complex)
    r12 = np.array([[c12, s12, 0], [-s12, c12, 0], [0, 0, 1]], dtype=complex)
    return r23 @ u13 @ r12


def masses(dm2_32: float, dm2_21: float, hierarchy: int) -> np.ndarray:
    return np.array([0.0, dm2_21, hierarchy * abs(dm2_32) + dm2_21])


def vacuum_prob(U: np.ndarray, m2: np.ndarray, L: float, E: float, a: int, b: int, antinu: bool) -> float:
    """Eq. 1.1 of the paper as read in DESIGN.md A1: |sum_i U*_{a i} U_{b i} exp(-i m_i^2 L / 2E)|^2."""
    Ue = U.conj() if antinu else U
    amp = sum(Ue[a, i].conjugate() * Ue[b, i] * np.exp(-1j * K_PHASE * m2[i] * L / E) for i in range(3))
    return float(abs(amp) ** 2)


def matter_term(rho: float, E: float, antinu: bool) -> float:
    A = K_MATTER * Y_E * rho * E
    return -A if antinu else A


def hamiltonian(U: np.ndarray, m2: np.ndarray, rho: float, E: float, antinu: bool) -> np.ndarray:
    """Flavour-basis H in eV^2 (used by the RK4 pin and the eigenvalue pin only)."""
    Ue = U.conj() if antinu else U
    H = Ue @ np.diag(m2).astype(complex) @ Ue.conj().T
    H[0, 0] += matter_term(rho, E, antinu)
    return H


def rk4_probs(H: np.ndarray, L: float, E: float, n_steps: int = 20000) -> np.ndarray:
    """Integrate i dpsi/dl = (K_PHASE / E) H psi from l = 0 to L for the three flavour initial states.
    Returns P[beta, alpha] = |psi_beta(L)|^2 starting from flavour alpha."""
    G = (-1j * K_PHASE / E) * H
    psi = np.eye(3, dtype=complex)      # column alpha = initial state alpha
    h = L / n_steps
    for _ in range(n_steps):
        k1 = G @ psi
        k2 = G @ (psi + 0.5 * h * k1)
        k3 = G @ (psi + 0.5 * h * k2)
        k4 = G @ (psi + h * k3)
        psi = psi + (h / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
    return np.abs(psi) ** 2


def two_flavour_survival(sin2_2theta: float, dm2: float, L: float, E: float) -> float:
    return 1.0 - sin2_2theta * math.sin(0.5 * K_PHASE * dm2 * L / E) ** 2


def msw_two_flavour(theta: float, dm2: float, A: float, L: float, E: float) -> float:
    """Transition probability sin^2(2 theta_M) sin^2(phase_M) of a two-level system with vacuum angle
    theta, splitting dm2 and matter term A (all eV^2)."""
    s2, c2 = math.sin(2 * theta), math.cos(2 * theta)
    C = math.sqrt((c2 - A / dm2) ** 2 + s2 ** 2)
    return (s2 / C) ** 2 * math.sin(0.5 * K_PHASE * dm2 * C * L / E) ** 2
