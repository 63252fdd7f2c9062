"""Thin ctypes binding of libosc_b200.so (include/osc.h): argument marshalling only.

Every function has the name of the C entry point it calls; all arithmetic of the path runs in the
CUDA kernels behind that call.  PyTorch supplies device memory (``tensor.data_ptr()``) and the stream
(``torch.cuda.current_stream()``) and nothing else.  There is no CPU fallback: if the shared library
is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
import threading
from typing import Mapping, Optional, Sequence

import numpy as np

from . import build as _build

_dp = ctypes.c_void_p
_lib: Optional[ctypes.CDLL] = None

N_CHANNELS = 4  # OSC_N_CHANNELS
PARAM_FIELDS = ("sin2_th12", "sin2_th23", "sin2_th13", "dm2_32", "dm2_21", "delta_cp", "rho_g_cm3",
                "L_km", "hierarchy")

# every symbol include/osc.h declares (tests/test_abi.py checks the header against this list)
EXPORTS = ("osc_set_params", "osc_prob", "osc_prob_all", "osc_reweight_bin", "osc_reweight_bin_scales", "osc_reweight_bin_batch",
           "osc_plan_create", "osc_plan_reweight_bin", "osc_plan_reweight_bin_batch", "osc_plan_destroy",
           "osc_neg2lnl", "osc_bin_centre_compare", "osc_bin_index", "osc_prob_host", "osc_reweight_bin_host", "osc_reweight_bin_scales_host", "osc_last_error", "osc_launch_count",
           "osc_version", "osc_set_device", "osc_get_device", "osc_fp64_peak_probe", "osc_set_batch_path",
           "osc_set_k2_tuning", "osc_fp64_issue_probe", "osc_reweight_bin_static")


class OscError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"libosc_b200 status {status}: {message}")
        self.status = status


class osc_params(ctypes.Structure):
    """Mirror of ``osc_params`` in include/osc.h."""
    _fields_ = [("sin2_th12", ctypes.c_double), ("sin2_th23", ctypes.c_double), ("sin2_th13", ctypes.c_double),
                ("dm2_32", ctypes.c_double), ("dm2_21", ctypes.c_double), ("delta_cp", ctypes.c_double),
                ("rho_g_cm3", ctypes.c_double), ("L_km", ctypes.c_double), ("hierarchy", ctypes.c_int)]


def lib() -> ctypes.CDLL:
    """Load libosc_b200.so (built in-tree by paper_1311_7579_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if not os.path.exists(path):
        raise OscError(-100, f"{path} is missing: run `python -m paper_1311_7579_b200.build` "
                             "(there is no CPU fallback)")
    L = ctypes.CDLL(path)
    d, i, sz, vp = ctypes.c_double, ctypes.c_int, ctypes.c_size_t, ctypes.c_void_p
    L.osc_set_params.argtypes = [d, d, d, d, d, d, d, d, i]
    L.osc_prob.argtypes = [_dp, sz, i, i, i, _dp, vp]
    L.osc_prob_all.argtypes = [_dp, sz, i, _dp, vp]
    L.osc_reweight_bin.argtypes = [_dp, _dp, _dp, _dp, sz, d, _dp, i, _dp, vp]
    L.osc_reweight_bin_scales.argtypes = [_dp, _dp, _dp, _dp, sz, ctypes.POINTER(d), i, _dp, i, _dp, vp]
    L.osc_reweight_bin_batch.argtypes = [ctypes.POINTER(osc_params), i, _dp, _dp, _dp, _dp, sz, d, _dp, i, _dp, vp]
    L.osc_bin_index.argtypes = [_dp, _dp, _dp, sz, d, _dp, i, _dp, vp]
    L.osc_neg2lnl.argtypes = [_dp, i, i, _dp, d, _dp, vp]
    L.osc_plan_create.argtypes = [_dp, _dp, _dp, _dp, sz, d, _dp, i, vp, ctypes.POINTER(vp)]
    L.osc_plan_reweight_bin.argtypes = [vp, _dp, vp]
    L.osc_plan_reweight_bin_batch.argtypes = [vp, ctypes.POINTER(osc_params), i, _dp, vp]
    L.osc_plan_destroy.argtypes = [vp]
    L.osc_bin_centre_compare.argtypes = [_dp, _dp, _dp, sz, _dp, i, _dp, _dp, vp]
    L.osc_prob_host.argtypes = [_dp, sz, i, i, i, _dp]
    L.osc_reweight_bin_host.argtypes = [_dp, _dp, _dp, _dp, sz, d, _dp, i, _dp]
    L.osc_reweight_bin_scales_host.argtypes = [_dp, _dp, _dp, _dp, sz, ctypes.POINTER(d), i, _dp, i, _dp]
    L.osc_set_device.argtypes = [i]
    L.osc_get_device.argtypes = [ctypes.POINTER(i)]
    L.osc_fp64_peak_probe.argtypes = [i, i, ctypes.POINTER(d), vp]
    L.osc_fp64_issue_probe.argtypes = [i, i, i, ctypes.POINTER(d), vp]
    L.osc_set_batch_path.argtypes = [ctypes.c_char_p]
    L.osc_set_k2_tuning.argtypes = [i, i, i, i]
    L.osc_reweight_bin_static.argtypes = [_dp, _dp, _dp, _dp, sz, d, _dp, i, _dp, vp]
    for name in ("osc_set_params", "osc_prob", "osc_prob_all", "osc_reweight_bin", "osc_reweight_bin_scales",
                 "osc_reweight_bin_batch",
                 "osc_plan_create", "osc_plan_reweight_bin", "osc_plan_reweight_bin_batch", "osc_plan_destroy",
                 "osc_neg2lnl", "osc_bin_centre_compare", "osc_bin_index", "osc_prob_host", "osc_reweight_bin_host", "osc_reweight_bin_scales_host", "osc_set_device",
                 "osc_get_device",
                 "osc_fp64_peak_probe", "osc_set_batch_path", "osc_set_k2_tuning", "osc_fp64_issue_probe",
                 "osc_reweight_bin_static"):
        getattr(L, name).restype = i
    L.osc_last_error.restype = ctypes.c_char_p
    L.osc_version.restype = ctypes.c_char_p
    L.osc_launch_count.restype = ctypes.c_ulonglong
    _lib = L
    return L


def _check(rc: int) -> None:
    if rc != 0:
        raise OscError(rc, lib().osc_last_error().decode())


def _stream(stream) -> int:
    import torch

    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _dev(t, dtype, what: str) -> int:
    """Device pointer of a contiguous CUDA tensor of the given dtype."""
    if not t.is_cuda:
        raise TypeError(f"{what} must be a CUDA tensor")
    if t.dtype != dtype:
        raise TypeError(f"{what} must have dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise TypeError(f"{what} must be contiguous")
    _sync_device(t.device.index)
    return t.data_ptr()


_tls = threading.local()       # the current CUDA device is a per-thread property, and so is this cache of it


def _sync_device(index: Optional[int]) -> None:
    """Align the library's (statically linked) CUDA runtime with the device of the tensors."""
    if index is None:
        index = 0
    if getattr(_tls, "dev", None) != index:
        _check(lib().osc_set_device(int(index)))
        _tls.dev = index


def _host(a: np.ndarray, dtype, what: str) -> int:
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
        raise TypeError(f"{what} must be a C-contiguous numpy array of dtype {np.dtype(dtype)}")
    return a.ctypes.data


def make_params(p) -> osc_params:
    if isinstance(p, osc_params):
        return p
    if isinstance(p, Mapping):
        return osc_params(*[p[f] if f != "hierarchy" else int(p[f]) for f in PARAM_FIELDS])
    return osc_params(*[getattr(p, f) if f != "hierarchy" else int(getattr(p, f)) for f in PARAM_FIELDS])


# ---------------------------------------------------------------------------------------------------
# entry points (same names and argument order as include/osc.h)
# ---------------------------------------------------------------------------------------------------

def osc_set_params(sin2_th12: float, sin2_th23: float, sin2_th13: float, dm2_32: float, dm2_21: float,
                   delta_cp: float, rho_g_cm3: float, L_km: float, hierarchy: int = 1) -> None:
    _check(lib().osc_set_params(sin2_th12, sin2_th23, sin2_th13, dm2_32, dm2_21, delta_cp, rho_g_cm3, L_km,
                                int(hierarchy)))


def osc_prob(E_true, flavour_in: int, flavour_out: int, antinu: int, P_out=None, stream=None):
    import torch

    n = E_true.numel()
    if P_out is None:
        P_out = torch.empty_like(E_true)
    if P_out.numel() != n:
        raise ValueError("P_out must hold n values")
    _check(lib().osc_prob(_dev(E_true, torch.float64, "E_true"), n, flavour_in, flavour_out, int(antinu),
                          _dev(P_out, torch.float64, "P_out"), _stream(stream)))
    return P_out


def osc_prob_all(E_true, antinu: int, P_out=None, stream=None):
    """[9, n] tensor, row 3*beta + alpha = P(alpha -> beta)."""
    import torch

    n = E_true.numel()
    if P_out is None:
        P_out = torch.empty((9, n), dtype=torch.float64, device=E_true.device)
    if P_out.numel() != 9 * n:
        raise ValueError("P_out must hold 9 * n values")
    _check(lib().osc_prob_all(_dev(E_true, torch.float64, "E_true"), n, int(antinu),
                              _dev(P_out, torch.float64, "P_out"), _stream(stream)))
    return P_out


def _event_ptrs(E_true, E_reco, w0, channel):
    import torch

    n = E_true.numel()
    if E_reco.numel() != n or channel.numel() != n or (w0 is not None and w0.numel() != n):
        raise ValueError("event arrays differ in length")
    return (n, _dev(E_true, torch.float64, "E_true"), _dev(E_reco, torch.float64, "E_reco"),
            _dev(w0, torch.float64, "w0") if w0 is not None else None, _dev(channel, torch.int8, "channel"))


def _n_bins(bin_edges) -> int:
    nb = (bin_edges.numel() if hasattr(bin_edges, "numel") else bin_edges.size) - 1
    if nb < 1:
        raise ValueError("bin_edges must hold at least two edges")
    return nb


def osc_reweight_bin(E_true, E_reco, w0, channel, energy_scale: float, bin_edges, hist_out=None, stream=None):
    """[N_CHANNELS, n_bins] histogram tensor (overwritten)."""
    import torch

    nb = _n_bins(bin_edges)
    n, pt, pr, pw, pc = _event_ptrs(E_true, E_reco, w0, channel)
    if hist_out is None:
        hist_out = torch.empty((N_CHANNELS, nb), dtype=torch.float64, device=E_true.device)
    if hist_out.numel() != N_CHANNELS * nb:
        raise ValueError("hist_out must hold N_CHANNELS * n_bins values")
    _check(lib().osc_reweight_bin(pt, pr, pw, pc, n, float(energy_scale), _dev(bin_edges, torch.float64, "bin_edges"),
                                  nb, _dev(hist_out, torch.float64, "hist_out"), _stream(stream)))
    return hist_out


def osc_reweight_bin_static(E_true, E_reco, w0, channel, energy_scale: float, bin_edges, hist_out, stream=None):
    """osc_reweight_bin without any allocation in the library (scratch in a static device array, at most 128 bins);
    the caller passes hist_out: this wrapper allocates nothing either."""
    import torch

    nb = _n_bins(bin_edges)
    n, pt, pr, pw, pc = _event_ptrs(E_true, E_reco, w0, channel)
    if hist_out.numel() != N_CHANNELS * nb:
        raise ValueError("hist_out must hold N_CHANNELS * n_bins values")
    _check(lib().osc_reweight_bin_static(pt, pr, pw, pc, n, float(energy_scale),
                                         _dev(bin_edges, torch.float64, "bin_edges"), nb,
                                         _dev(hist_out, torch.float64, "hist_out"), _stream(stream)))
    return hist_out


def osc_reweight_bin_scales(E_true, E_reco, w0, channel, energy_scales: Sequence[float], bin_edges, hist_out=None,
                            stream=None):
    """[n_scales, N_CHANNELS, n_bins] histograms, one slice per energy-scale value, in one pass over the events."""
    import torch

    nb = _n_bins(bin_edges)
    n, pt, pr, pw, pc = _event_ptrs(E_true, E_reco, w0, channel)
    ns = len(energy_scales)
    arr = (ctypes.c_double * max(ns, 1))(*[float(v) for v in energy_scales])
    if hist_out is None:
        hist_out = torch.empty((ns, N_CHANNELS, nb), dtype=torch.float64, device=E_true.device)
    if hist_out.numel() != ns * N_CHANNELS * nb:
        raise ValueError("hist_out must hold n_scales * N_CHANNELS * n_bins values")
    _check(lib().osc_reweight_bin_scales(pt, pr, pw, pc, n, arr, ns, _dev(bin_edges, torch.float64, "bin_edges"), nb,
                                         _dev(hist_out, torch.float64, "hist_out"), _stream(stream)))
    return hist_out


def pack_params(points: Sequence):
    """The osc_params array of a list of parameter sets (marshalling only).  osc_reweight_bin_batch takes either
    the list or this array; a caller that scans the same points repeatedly packs them once."""
    return (osc_params * max(len(points), 1))(*[make_params(q) for q in points])


def osc_reweight_bin_batch(points: Sequence, E_true, E_reco, w0, channel, energy_scale: float, bin_edges,
                           hist_out=None, stream=None):
    """[n_points, N_CHANNELS, n_bins] histograms, one slice per parameter set, in one call."""
    import torch

    nb = _n_bins(bin_edges)
    n, pt, pr, pw, pc = _event_ptrs(E_true, E_reco, w0, channel)
    npts = len(points)
    arr = points if isinstance(points, ctypes.Array) else pack_params(points)
    if hist_out is None:
        hist_out = torch.empty((npts, N_CHANNELS, nb), dtype=torch.float64, device=E_true.device)
    if hist_out.numel() != npts * N_CHANNELS * nb:
        raise ValueError("hist_out must hold n_points * N_CHANNELS * n_bins values")
    _check(lib().osc_reweight_bin_batch(arr, npts, pt, pr, pw, pc, n, float(energy_scale),
                                        _dev(bin_edges, torch.float64, "bin_edges"), nb,
                                        _dev(hist_out, torch.float64, "hist_out"), _stream(stream)))
    return hist_out


class OscPlan:
    """Handle of an ``osc_plan`` (include/osc.h) plus what the binding needs to size outputs.  Destroyed with
    ``osc_plan_destroy`` (or when the object is collected)."""

    def __init__(self, ptr: int, n_bins: int, device):
        self.ptr, self.n_bins, self.device = ptr, n_bins, device

    def __del__(self):
        try:
            osc_plan_destroy(self)
        except Exception:
            pass


def osc_plan_create(E_true, E_reco, w0, channel, energy_scale: float, bin_edges, stream=None) -> OscPlan:
    import torch

    nb = _n_bins(bin_edges)
    n, pt, pr, pw, pc = _event_ptrs(E_true, E_reco, w0, channel)
    out = ctypes.c_void_p()
    _check(lib().osc_plan_create(pt, pr, pw, pc, n, float(energy_scale), _dev(bin_edges, torch.float64, "bin_edges"), nb,
                                 _stream(stream), ctypes.byref(out)))
    return OscPlan(out.value, nb, E_true.device)


def osc_plan_reweight_bin(plan: OscPlan, hist_out=None, stream=None):
    """[N_CHANNELS, n_bins] histogram of the planned events with the parameters of osc_set_params."""
    import torch

    if hist_out is None:
        hist_out = torch.empty((N_CHANNELS, plan.n_bins), dtype=torch.float64, device=plan.device)
    if hist_out.numel() != N_CHANNELS * plan.n_bins:
        raise ValueError("hist_out must hold N_CHANNELS * n_bins values")
    _check(lib().osc_plan_reweight_bin(plan.ptr, _dev(hist_out, torch.float64, "hist_out"), _stream(stream)))
    return hist_out


def osc_plan_reweight_bin_batch(plan: OscPlan, points: Sequence, hist_out=None, stream=None):
    """[n_points, N_CHANNELS, n_bins] histograms of the planned events, one slice per parameter set."""
    import torch

    npts = len(points)
    arr = points if isinstance(points, ctypes.Array) else pack_params(points)
    if hist_out is None:
        hist_out = torch.empty((npts, N_CHANNELS, plan.n_bins), dtype=torch.float64, device=plan.device)
    if hist_out.numel() != npts * N_CHANNELS * plan.n_bins:
        raise ValueError("hist_out must hold n_points * N_CHANNELS * n_bins values")
    _check(lib().osc_plan_reweight_bin_batch(plan.ptr, arr, npts, _dev(hist_out, torch.float64, "hist_out"),
                                             _stream(stream)))
    return hist_out


def osc_plan_destroy(plan: OscPlan) -> None:
    if plan is not None and plan.ptr:
        ptr, plan.ptr = plan.ptr, None
        _check(lib().osc_plan_destroy(ptr))


def osc_neg2lnl(hist, data, norm: float = 1.0, out=None, stream=None):
    """[n_points] tensor of -2 ln lambda (Poisson likelihood ratio) of hist[p] * norm against data."""
    import torch

    n_cells = data.numel()
    if n_cells == 0 or hist.numel() % n_cells != 0:
        raise ValueError("hist must hold n_points * data.numel() values")
    npts = hist.numel() // n_cells
    if out is None:
        out = torch.empty(npts, dtype=torch.float64, device=hist.device)
    if out.numel() != npts:
        raise ValueError("out must hold n_points values")
    _check(lib().osc_neg2lnl(_dev(hist, torch.float64, "hist"), npts, n_cells, _dev(data, torch.float64, "data"),
                             float(norm), _dev(out, torch.float64, "out"), _stream(stream)))
    return out


def osc_bin_centre_compare(E_true, w0, channel, bin_edges, stream=None):
    """(hist_event, hist_centre), each [N_CHANNELS, n_bins], over TRUE-energy bins (include/osc.h)."""
    import torch

    n, pt, _, pw, pc = _event_ptrs(E_true, E_true, w0, channel)
    nb = _n_bins(bin_edges)
    he = torch.empty((N_CHANNELS, nb), dtype=torch.float64, device=E_true.device)
    hc = torch.empty_like(he)
    _check(lib().osc_bin_centre_compare(pt, pw, pc, n, _dev(bin_edges, torch.float64, "bin_edges"), nb,
                                        _dev(he, torch.float64, "hist_event_out"),
                                        _dev(hc, torch.float64, "hist_centre_out"), _stream(stream)))
    return he, hc


def osc_bin_index(E_true, E_reco, channel, energy_scale: float, bin_edges, bin_out=None, stream=None):
    import torch

    nb = _n_bins(bin_edges)
    if bin_out is not None and bin_out.numel() != E_true.numel():
        raise ValueError("bin_out must hold n values")
    n, pt, pr, _, pc = _event_ptrs(E_true, E_reco, None, channel)
    if bin_out is None:
        bin_out = torch.empty(n, dtype=torch.int32, device=E_true.device)
    _check(lib().osc_bin_index(pt, pr, pc, n, float(energy_scale), _dev(bin_edges, torch.float64, "bin_edges"), nb,
                               _dev(bin_out, torch.int32, "bin_out"), _stream(stream)))
    return bin_out


def osc_prob_host(E_true: np.ndarray, flavour_in: int, flavour_out: int, antinu: int,
                  P_out: Optional[np.ndarray] = None) -> np.ndarray:
    """Host buffers in and out (the flow of the paper's Listing 1): H2D, kernel, D2H, synchronise."""
    if P_out is None:
        P_out = np.empty_like(E_true)
    if P_out.size != E_true.size:
        raise ValueError("P_out must hold n values")
    _check(lib().osc_prob_host(_host(E_true, np.float64, "E_true"), E_true.size, flavour_in, flavour_out,
                               int(antinu), _host(P_out, np.float64, "P_out")))
    return P_out


def osc_reweight_bin_host(E_true: np.ndarray, E_reco: np.ndarray, w0: np.ndarray, channel: np.ndarray,
                          energy_scale: float, bin_edges: np.ndarray,
                          hist_out: Optional[np.ndarray] = None) -> np.ndarray:
    nb = _n_bins(bin_edges)
    if hist_out is None:
        hist_out = np.empty((N_CHANNELS, nb), dtype=np.float64)
    _check_host_events(E_true, E_reco, w0, channel)
    if hist_out.size != N_CHANNELS * nb:
        raise ValueError("hist_out must hold N_CHANNELS * n_bins values")
    _check(lib().osc_reweight_bin_host(_host(E_true, np.float64, "E_true"), _host(E_reco, np.float64, "E_reco"),
                                       _host(w0, np.float64, "w0"), _host(channel, np.int8, "channel"), E_true.size,
                                       float(energy_scale), _host(bin_edges, np.float64, "bin_edges"), nb,
                                       _host(hist_out, np.float64, "hist_out")))
    return hist_out


def _check_host_events(E_true, E_reco, w0, channel) -> None:
    n = E_true.size
    if E_reco.size != n or w0.size != n or channel.size != n:
        raise ValueError("host event arrays differ in length")


def osc_set_batch_path(path: str) -> None:
    """"auto" | "k2" | "k4" | "k4s" | "k4c" | "k5": code path of the batched calls (measurements and tests)."""
    _check(lib().osc_set_batch_path(path.encode()))


def osc_set_k2_tuning(threads: int = 0, slots: int = 0, n_sub: int = 0, blocks_per_sm: int = 0) -> None:
    """Launch shape of osc_reweight_bin's kernel; 0 leaves a field to the library (measurements and tests)."""
    _check(lib().osc_set_k2_tuning(int(threads), int(slots), int(n_sub), int(blocks_per_sm)))


def osc_last_error() -> str:
    return lib().osc_last_error().decode()


def osc_launch_count() -> int:
    return int(lib().osc_launch_count())


def osc_version() -> str:
    return lib().osc_version().decode()


def osc_set_device(device: int) -> None:
    _check(lib().osc_set_device(int(device)))
    _tls.dev = int(device)


def osc_get_device() -> int:
    v = ctypes.c_int(-1)
    _check(lib().osc_get_device(ctypes.byref(v)))
    return v.value


def osc_fp64_peak_probe(iters: int, blocks_per_sm: int = 4, stream=None) -> float:
    """Enqueue one DFMA-probe launch; returns its floating-point operation count."""
    flops = ctypes.c_double(0.0)
    _check(lib().osc_fp64_peak_probe(int(iters), int(blocks_per_sm), ctypes.byref(flops), _stream(stream)))
    return flops.value


def osc_fp64_issue_probe(kind: int, iters: int, blocks_per_sm: int = 4, stream=None) -> float:
    """Enqueue one launch of issue-probe `kind` (include/osc.h); returns its fp64 thread-instruction count."""
    cnt = ctypes.c_double(0.0)
    _check(lib().osc_fp64_issue_probe(int(kind), int(iters), int(blocks_per_sm), ctypes.byref(cnt), _stream(stream)))
    return cnt.value


def osc_reweight_bin_scales_host(E_true: np.ndarray, E_reco: np.ndarray, w0: np.ndarray, channel: np.ndarray,
                                 energy_scales: Sequence[float], bin_edges: np.ndarray,
                                 hist_out: Optional[np.ndarray] = None) -> np.ndarray:
    """Host buffers in and out, several energy scales, one trip of the events over PCIe."""
    nb = _n_bins(bin_edges)
    ns = len(energy_scales)
    if hist_out is None:
        hist_out = np.empty((ns, N_CHANNELS, nb), dtype=np.float64)
    arr = (ctypes.c_double * max(ns, 1))(*[float(v) for v in energy_scales])
    _check_host_events(E_true, E_reco, w0, channel)
    if hist_out.size != ns * N_CHANNELS * nb:
        raise ValueError("hist_out must hold n_scales * N_CHANNELS * n_bins values")
    _check(lib().osc_reweight_bin_scales_host(_host(E_true, np.float64, "E_true"), _host(E_reco, np.float64, "E_reco"),
                                              _host(w0, np.float64, "w0"), _host(channel, np.int8, "channel"),
                                              E_true.size, arr, ns, _host(bin_edges, np.float64, "bin_edges"), nb,
                                              _host(hist_out, np.float64, "hist_out")))
    return hist_out
