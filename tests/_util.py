"""Shared test helpers: compare fields, keep a record of the measured parity errors."""
from __future__ import annotations

import json
import os
from pathlib import Path

import numpy as np

from oracle import oracle_from_workload  # noqa: F401  (re-exported for the tests)

ROOT = Path(__file__).resolve().parent.parent

FIELD_GROUPS = {
    "E": ("Ex", "Ey", "Ez"),
    "H": ("Hx", "Hy", "Hz"),
    "M": ("Mxx", "Mxy", "Mxz", "Myx", "Myy", "Myz", "Mzx", "Mzy", "Mzz"),
}


def rel_linf(got: dict, ref: dict, group: str) -> float:
    """max |got-ref| over all components of the vector field / max |ref|  (A21)."""
    names = FIELD_GROUPS[group]
    num = max(float(np.max(np.abs(got[n] - ref[n]))) for n in names)
    den = max(float(np.max(np.abs(ref[n]))) for n in names)
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return num / den


def rel_linf_of_change(got: dict, ref: dict, ref0: dict, group: str = "M") -> float:
    """max |got-ref| / max |ref - ref0|: the error measured against how far the field MOVED during
    the run.  M turns by < 0.1 rad in any of the configs, so parity on M is a
    test of small differences; this figure is the one a slip in the damping or anisotropy term
    would show up in."""
    names = FIELD_GROUPS[group]
    num = max(float(np.max(np.abs(got[n] - ref[n]))) for n in names)
    den = max(float(np.max(np.abs(ref[n] - ref0[n]))) for n in names)
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return num / den


def record_parity(entry: dict) -> None:
    """Append one measured parity figure to the record (JSON lines).  The GPU suite writes it under
    gpurun_out/ (the folder that comes back from the GPU box); the summary committed under
    profiles/ is made from it."""
    path = Path(os.environ.get("FDTD_LLG_PARITY_RECORD", ROOT / "gpurun_out" / "parity_record.jsonl"))
    try:
        path.parent.mkdir(parents=True, exist_ok=True)
        with open(path, "a") as f:
            f.write(json.dumps(entry) + "\n")
    except OSError:
        pass
