"""Operation counts behind the roofline figures of bench.py: ``profiles/opcounts.json`` and its consistency check.

The roofline fractions bench.py prints are ``achieved = (counted fp64 operations per unit) x units / time``.  The
counts are not typed into bench.py: they are read from ``profiles/opcounts.json``, which this module writes from the
unedited ncu logs under ``profiles/`` (``smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum``,
``smsp__inst_executed.sum``, ``dram__bytes_{read,write}.sum`` per launch) together with the SHA-256 of every source
file the counted kernel includes.  ``stale()`` recomputes those hashes: if a kernel source has changed since the
capture, bench.py prints no fraction for that kernel (``roofline.frac = null``, ``counts_stale = true``) and
``tests/test_opcounts.py`` fails, so a stale constant cannot produce a number.

    python -m paper_1311_7579_b200.opcounts --write          # after new captures: rewrite profiles/opcounts.json
    python -m paper_1311_7579_b200.opcounts --check          # exit 1 if a counted kernel's sources have changed

No arithmetic of the method lives here.
"""
from __future__ import annotations

import csv
import hashlib
import io
import json
import os
import re
import subprocess
import sys
from typing import Dict, List

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
JSON_PATH = os.path.join(ROOT, "profiles", "opcounts.json")

_CORE = ["osc_core.cuh", "osc_math.cuh", "osc_coeffs.h", "osc_types.h", "osc_smem.cuh"]
_EVENT = _CORE + ["osc_kernels.cuh", "osc_bins.cuh", "osc_hist.cuh"]
_SCAN = _CORE + ["osc_scan.cuh", "osc_bins.cuh"]

# key -> how to read one capture.  `csv`: unedited ncu log under profiles/; `kernels`: regex over the kernel names whose
# launches are summed (one CALL of the library may be several launches); `calls`: how many calls the log holds (its
# sums are divided by it); `units`: units of work per call; `files`: sources the counted kernels include.
CAPTURES: Dict[str, dict] = {
    "k2": dict(csv="r2_k2_ops.csv", kernels=r"reweight_bin_kernel", calls=1, units=10_000_000, unit="event",
               files=_EVENT, what="osc_reweight_bin, 1e7 events, 50 bins (configs[2])"),
    "k2s": dict(csv="r2_k2s_ops.csv", kernels=r"reweight_bin_scales_kernel", calls=1, units=10_000_000, unit="event (3 scales)",
                files=_EVENT, what="osc_reweight_bin_scales, 1e7 events x 3 energy scales"),
    "k1": dict(csv="r2_k1_ops.csv", kernels=r"prob_kernel", calls=2, units=100_000, unit="event",
               files=_EVENT, what="osc_prob, 1e5 events, mu->mu and mu->e (configs[0]); mean of the two launches"),
    "k1b": dict(csv="r2_k1b_ops.csv", kernels=r"prob_all_kernel", calls=1, units=10_000_000, unit="event",
                files=_EVENT, what="osc_prob_all, 1e7 events, 9 outputs (configs[1])"),
    "k4": dict(csv="r2_k4_ops.csv", kernels=r"scan_|sort_", calls=1, units=1_000_000 * 1024, unit="(event, point)",
               files=_SCAN, what="osc_reweight_bin_batch, 1e6 events x 1024 grid points, all kernels of one call (configs[3])"),
    "k5": dict(csv="r2_k5_ops.csv", kernels=r"scan_|sort_", calls=1, units=1_000_000 * 1024, unit="(event, point)",
               files=_SCAN, what="the same call forced through k5 (osc_set_batch_path), all kernels of one call"),
    "plan": dict(csv="r2_plan_ops.csv", kernels=r"scan_full_one_kernel", calls=1, units=10_000_000, unit="event",
                 files=_SCAN, what="osc_plan_reweight_bin, 1e7 pre-sorted events (main kernel)"),
}

_M = {"dfma": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
      "dmul": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
      "dadd": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
      "warp_inst": "smsp__inst_executed.sum",
      "dram_read": "dram__bytes_read.sum", "dram_write": "dram__bytes_write.sum", "ns": "gpu__time_duration.sum"}


def file_hashes(files: List[str]) -> Dict[str, str]:
    out = {}
    for f in sorted(set(files)):
        with open(os.path.join(CSRC, f), "rb") as fh:
            out[f] = hashlib.sha256(fh.read()).hexdigest()
    return out


def read_ncu_csv(path: str) -> List[dict]:
    """One dict per profiled launch: kernel name, grid, block and the metric values (floats)."""
    txt = open(path).read()
    rows = list(csv.DictReader(io.StringIO(txt[txt.index('"ID"'):])))
    launches: Dict[str, dict] = {}
    for r in rows:
        d = launches.setdefault(r["ID"], {"kernel": r["Kernel Name"], "grid": r["Grid Size"], "block": r["Block Size"]})
        try:
            d[r["Metric Name"]] = float(r["Metric Value"].replace(",", ""))
        except ValueError:
            pass
    return [launches[k] for k in sorted(launches, key=int)]


def summarise(key: str, cap: dict, csv_dir: str) -> dict:
    launches = [l for l in read_ncu_csv(os.path.join(csv_dir, cap["csv"])) if re.search(cap["kernels"], l["kernel"])]
    if not launches:
        raise SystemExit(f"{cap['csv']}: no launch matches {cap['kernels']}")
    tot = {k: sum(l.get(m, 0.0) for l in launches) / cap["calls"] for k, m in _M.items()}
    u = float(cap["units"])
    fp64 = tot["dfma"] + tot["dmul"] + tot["dadd"]
    return {
        "what": cap["what"], "source": "profiles/" + cap["csv"], "unit": cap["unit"], "units_per_call": cap["units"],
        "launches_per_call": len(launches) // cap["calls"],
        "kernels": sorted({re.sub(r"\(.*", "", l["kernel"]).replace("void ", "") + " grid " + l["grid"] + " block " + l["block"]
                           for l in launches}),
        "dfma_per_unit": tot["dfma"] / u, "dmul_per_unit": tot["dmul"] / u, "dadd_per_unit": tot["dadd"] / u,
        "fp64_inst_per_unit": fp64 / u, "flop_per_unit": (2.0 * tot["dfma"] + tot["dmul"] + tot["dadd"]) / u,
        "inst_per_unit": 32.0 * tot["warp_inst"] / u,
        "dram_bytes_per_call": tot["dram_read"] + tot["dram_write"], "us_under_ncu": tot["ns"] * 1e-3,
        "files": file_hashes(cap["files"]),
    }


def write(csv_dir: str = os.path.join(ROOT, "profiles")) -> dict:
    try:
        commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    except OSError:
        commit = ""
    doc = {"comment": "written by `python -m paper_1311_7579_b200.opcounts --write` from the ncu logs named in `source`; "
                      "`files` are SHA-256 of the kernel sources at capture time (the commit below, plus the working tree)",
           "commit": commit, "kernels": {}}
    for key, cap in CAPTURES.items():
        if os.path.exists(os.path.join(csv_dir, cap["csv"])):
            doc["kernels"][key] = summarise(key, cap, csv_dir)
    with open(JSON_PATH, "w") as f:
        json.dump(doc, f, indent=1, sort_keys=True)
        f.write("\n")
    return doc


def load() -> dict:
    with open(JSON_PATH) as f:
        return json.load(f)


def stale(key: str, doc: dict = None) -> List[str]:
    """Names of the source files of kernel `key` that differ from the capture (empty list: the counts are current)."""
    doc = doc or load()
    k = doc["kernels"][key]
    now = file_hashes(list(k["files"]))
    return [f for f, h in k["files"].items() if now.get(f) != h]


def counts(key: str, doc: dict = None) -> dict:
    """The entry of kernel `key` with `stale` (list of changed files) and `commit` added."""
    doc = doc or load()
    k = dict(doc["kernels"][key])
    k["stale"] = stale(key, doc)
    k["commit"] = doc.get("commit", "")
    k.pop("files", None)
    return k


if __name__ == "__main__":
    if "--write" in sys.argv:
        d = write()
        for key, k in d["kernels"].items():
            print(f"{key:5s} {k['flop_per_unit']:9.2f} flop  {k['fp64_inst_per_unit']:8.2f} fp64  {k['inst_per_unit']:8.2f} inst per "
                  f"{k['unit']}; DRAM {k['dram_bytes_per_call'] / 1e6:.1f} MB per call")
    elif "--check" in sys.argv:
        doc = load()
        bad = {k: stale(k, doc) for k in doc["kernels"]}
        bad = {k: v for k, v in bad.items() if v}
        print("stale:" if bad else "opcounts.json is current", bad if bad else "")
        sys.exit(1 if bad else 0)
    else:
        print(__doc__)
