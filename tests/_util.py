"""Shared test helpers: run a Workload on the oracle / the CUDA library, compare fields."""
from __future__ import annotations

import numpy as np

from oracle import Oracle

FIELD_GROUPS = {
    "E": ("Ex", "Ey", "Ez"),
    "H": ("Hx", "Hy", "Hz"),
    "M": ("Mxx", "Mxy", "Mxz", "Myx", "Myy", "Myz", "Mzx", "Mzy", "Mzz"),
}


def oracle_from_workload(w, kind="f64", time_scheme=0) -> Oracle:
    a = w.numpy()
    m = a["materials"]
    o = Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.dt,
               eps_r=m.get("eps_r"), sigma=m.get("sigma"), mu_r=m.get("mu_r"),
               Ms=m.get("Ms"), alpha=m.get("alpha"), gamma=m.get("gamma"),
               bc=w.bc, enable_llg=w.enable_llg, h_bias=w.h_bias, ani_hk=w.ani_hk,
               ani_axis=w.ani_axis, llg_tol=w.llg_tol, llg_max_iter=w.llg_max_iter, kind=kind,
               time_scheme=time_scheme, pml=getattr(w, "pml", None),
               **{k: getattr(w, k) for k in ("pml_r0", "pml_order") if getattr(w, k, None) is not None})
    o.set_fields(a["E"], a["H"], a["M_cell"])
    for s in w.sources:
        prof = None if s.profile is None else s.profile.detach().cpu().numpy()
        o.set_source(s.comp, s.lo, s.hi, prof, s.amplitude, s.f0, s.t0, s.tp, kind=getattr(s, "kind", 0))
    return o


def rel_linf(got: dict, ref: dict, group: str) -> float:
    """max |got-ref| over all components of the vector field / max |ref|  (A21)."""
    names = FIELD_GROUPS[group]
    num = max(float(np.max(np.abs(got[n] - ref[n]))) for n in names)
    den = max(float(np.max(np.abs(ref[n]))) for n in names)
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return num / den
