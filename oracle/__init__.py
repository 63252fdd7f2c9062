"""ctypes loader for the CPU oracle (oracle/osc_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_1311_7579_b200`` and the product imports nothing from here.

The functions take and return host numpy arrays; every value is computed by the C
oracle (long double, Jacobi eigen-decomposition; see the header of osc_oracle.c).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "osc_oracle.c")
_LIB = os.path.join(_HERE, "liboscoracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, long double, OpenMP, no FP contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _CParams(ctypes.Structure):
    _fields_ = [("sin2_th12", ctypes.c_double), ("sin2_th23", ctypes.c_double),
                ("sin2_th13", ctypes.c_double), ("dm2_32", ctypes.c_double),
                ("dm2_21", ctypes.c_double), ("delta_cp", ctypes.c_double),
                ("rho_g_cm3", ctypes.c_double), ("L_km", ctypes.c_double),
                ("hierarchy", ctypes.c_int)]


@dataclass(frozen=True)
class Params:
    """One oscillation-parameter set; fields and order of ``osc_set_params`` (north_star)."""
    sin2_th12: float
    sin2_th23: float
    sin2_th13: float
    dm2_32: float
    dm2_21: float
    delta_cp: float
    rho_g_cm3: float
    L_km: float
    hierarchy: int = 1

    def _c(self) -> _CParams:
        return _CParams(self.sin2_th12, self.sin2_th23, self.sin2_th13, self.dm2_32, self.dm2_21,
                        self.delta_cp, self.rho_g_cm3, self.L_km, int(self.hierarchy))


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_i8p = ctypes.POINTER(ctypes.c_int8)
_i32p = ctypes.POINTER(ctypes.c_int32)


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        P = ctypes.POINTER(_CParams)
        _lib.oracle_prob.argtypes = [P, _dp, ctypes.c_size_t, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp]
        _lib.oracle_prob_all.argtypes = [P, _dp, ctypes.c_size_t, ctypes.c_int, _dp]
        _lib.oracle_evolution.argtypes = [P, ctypes.c_double, ctypes.c_int, _dp]
        _lib.oracle_eigenvalues.argtypes = [P, ctypes.c_double, ctypes.c_int, _dp]
        _lib.oracle_bin_index.argtypes = [_dp, _dp, _i8p, ctypes.c_size_t, ctypes.c_double, _dp,
                                          ctypes.c_int, _i32p]
        _lib.oracle_reweight_bin.argtypes = [P, _dp, _dp, _dp, _i8p, ctypes.c_size_t, ctypes.c_double,
                                             _dp, ctypes.c_int, _dp]
        _lib.oracle_reweight_bin_batch.argtypes = [P, ctypes.c_int, _dp, _dp, _dp, _i8p, ctypes.c_size_t,
                                                   ctypes.c_double, _dp, ctypes.c_int, _dp]
        _lib.oracle_bin_centre_compare.argtypes = [P, _dp, _dp, _i8p, ctypes.c_size_t, _dp, ctypes.c_int, _dp, _dp]
        _lib.oracle_bin_centre_compare.restype = ctypes.c_int
        _lib.oracle_neg2lnl.argtypes = [_dp, ctypes.c_int, ctypes.c_int, _dp, ctypes.c_double, _dp]
        _lib.oracle_neg2lnl.restype = ctypes.c_int
        _lib.oracle_set_threads.argtypes = [ctypes.c_int]
        for f in ("oracle_prob", "oracle_prob_all", "oracle_evolution", "oracle_eigenvalues",
                  "oracle_bin_index", "oracle_reweight_bin", "oracle_reweight_bin_batch",
                  "oracle_n_channels", "oracle_threads"):
            getattr(_lib, f).restype = ctypes.c_int
        _lib.oracle_set_threads.restype = None
    return _lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a: np.ndarray, t=_dp):
    return a.ctypes.data_as(t)


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise ValueError(f"{what} failed with status {rc}")


def n_channels() -> int:
    return lib().oracle_n_channels()


def threads() -> int:
    """Number of OpenMP threads the oracle's event loops will use."""
    return lib().oracle_threads()


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def prob(p: Params, E, fl_in: int, fl_out: int, antinu: int) -> np.ndarray:
    E = _f64(E)
    out = np.empty_like(E)
    c = p._c()
    _check(lib().oracle_prob(ctypes.byref(c), _ptr(E), E.size, fl_in, fl_out, int(antinu), _ptr(out)),
           "oracle_prob")
    return out


def prob_all(p: Params, E, antinu: int) -> np.ndarray:
    """[9, n] array, row 3*beta + alpha = P(alpha -> beta)."""
    E = _f64(E)
    out = np.empty((9, E.size), dtype=np.float64)
    c = p._c()
    _check(lib().oracle_prob_all(ctypes.byref(c), _ptr(E), E.size, int(antinu), _ptr(out)), "oracle_prob_all")
    return out


def evolution(p: Params, E: float, antinu: int) -> np.ndarray:
    """Complex 3x3 S, S[beta, alpha]."""
    out = np.empty(18, dtype=np.float64)
    c = p._c()
    _check(lib().oracle_evolution(ctypes.byref(c), float(E), int(antinu), _ptr(out)), "oracle_evolution")
    return (out[0::2] + 1j * out[1::2]).reshape(3, 3)


def eigenvalues(p: Params, E: float, antinu: int) -> np.ndarray:
    out = np.empty(3, dtype=np.float64)
    c = p._c()
    _check(lib().oracle_eigenvalues(ctypes.byref(c), float(E), int(antinu), _ptr(out)), "oracle_eigenvalues")
    return out


def bin_index(E_true, E_reco, channel, energy_scale: float, edges) -> np.ndarray:
    E_true, E_reco, edges = _f64(E_true), _f64(E_reco), _f64(edges)
    channel = np.ascontiguousarray(channel, dtype=np.int8)
    out = np.empty(E_true.size, dtype=np.int32)
    _check(lib().oracle_bin_index(_ptr(E_true), _ptr(E_reco), _ptr(channel, _i8p), E_true.size,
                                  float(energy_scale), _ptr(edges), edges.size - 1, _ptr(out, _i32p)),
           "oracle_bin_index")
    return out


def reweight_bin(p: Params, E_true, E_reco, w0, channel, energy_scale: float, edges) -> np.ndarray:
    """[n_channels, n_bins] histogram."""
    E_true, E_reco, w0, edges = _f64(E_true), _f64(E_reco), _f64(w0), _f64(edges)
    channel = np.ascontiguousarray(channel, dtype=np.int8)
    nb = edges.size - 1
    out = np.empty((n_channels(), nb), dtype=np.float64)
    c = p._c()
    _check(lib().oracle_reweight_bin(ctypes.byref(c), _ptr(E_true), _ptr(E_reco), _ptr(w0),
                                     _ptr(channel, _i8p), E_true.size, float(energy_scale),
                                     _ptr(edges), nb, _ptr(out)), "oracle_reweight_bin")
    return out


def reweight_bin_batch(points, E_true, E_reco, w0, channel, energy_scale: float, edges) -> np.ndarray:
    """[n_points, n_channels, n_bins] histograms."""
    E_true, E_reco, w0, edges = _f64(E_true), _f64(E_reco), _f64(w0), _f64(edges)
    channel = np.ascontiguousarray(channel, dtype=np.int8)
    nb = edges.size - 1
    arr = (_CParams * len(points))(*[q._c() for q in points])
    out = np.empty((len(points), n_channels(), nb), dtype=np.float64)
    _check(lib().oracle_reweight_bin_batch(arr, len(points), _ptr(E_true), _ptr(E_reco), _ptr(w0),
                                           _ptr(channel, _i8p), E_true.size, float(energy_scale),
                                           _ptr(edges), nb, _ptr(out)), "oracle_reweight_bin_batch")
    return out


def neg2lnl(hist, data, norm: float = 1.0) -> np.ndarray:
    """[n_points] values of the Poisson likelihood ratio -2 ln lambda of norm * hist[p] against data."""
    data = _f64(data).ravel()
    hist = _f64(hist).reshape(-1, data.size)
    out = np.empty(hist.shape[0], dtype=np.float64)
    _check(lib().oracle_neg2lnl(_ptr(hist), hist.shape[0], data.size, _ptr(data), float(norm), _ptr(out)),
           "oracle_neg2lnl")
    return out


def bin_centre_compare(p: Params, E_true, w0, channel, edges):
    """(hist_event, hist_centre), each [n_channels, n_bins], over TRUE-energy bins."""
    E_true, w0, edges = _f64(E_true), _f64(w0), _f64(edges)
    channel = np.ascontiguousarray(channel, dtype=np.int8)
    nb = edges.size - 1
    he = np.empty((n_channels(), nb), dtype=np.float64)
    hc = np.empty_like(he)
    c = p._c()
    _check(lib().oracle_bin_centre_compare(ctypes.byref(c), _ptr(E_true), _ptr(w0), _ptr(channel, _i8p), E_true.size,
                                           _ptr(edges), nb, _ptr(he), _ptr(hc)), "oracle_bin_centre_compare")
    return he, hc
