"""ctypes loader for ``fdtd_llg_oracle.c`` -- TEST INFRASTRUCTURE (see the C file's header).

Builds two shared objects next to this file:

* ``liboracle_f64.so``  REAL = double, increment-form LLG solve: the parity reference.
* ``liboracle_ld.so``   REAL = long double, eqs. 18-21 exactly as printed:
  the fidelity cross-check for the increment form (reading A24).

Both are compiled ``-O2 -ffp-contract=off`` (no FMA contraction, no reassociation) with
OpenMP over k; every loop is Jacobi-style, so threading does not change a single bit.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fdtd_llg_oracle.c"
_LIBS = {
    "f64": (_HERE / "liboracle_f64.so", ["-DORC_PREFIX=oracle_"], "oracle_"),
    "ld": (
        _HERE / "liboracle_ld.so",
        ["-DORACLE_LITERAL", "-DREAL=long double", "-DORC_PREFIX=oracle_ld_"],
        "oracle_ld_",
    ),
}
_loaded: dict[str, C.CDLL] = {}


def build_oracle(force: bool = False) -> None:
    """Compile both builds of the oracle with gcc (no-op when up to date)."""
    for _, (lib, defs, _) in _LIBS.items():
        if not force and lib.exists() and lib.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               *defs, str(_SRC), "-o", str(lib), "-lm"]
        subprocess.run(cmd, check=True)


def _lib(kind: str) -> tuple[C.CDLL, str]:
    path, _, prefix = _LIBS[kind]
    if kind not in _loaded:
        build_oracle()
        _loaded[kind] = C.CDLL(str(path))
    return _loaded[kind], prefix


_DP = C.POINTER(C.c_double)
_IP = C.POINTER(C.c_int)


def _dptr(a):
    return None if a is None else a.ctypes.data_as(_DP)


def _as_f64(a, n):
    if a is None:
        return None
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1))
    if a.size != n:
        raise ValueError(f"array has {a.size} entries, expected {n}")
    return a


def constants(kind: str = "f64") -> dict:
    lib, p = _lib(kind)
    out = (C.c_double * 3)()
    getattr(lib, p + "constants")(out)
    return {"mu0": out[0], "eps0": out[1], "c0": out[2]}


class Oracle:
    """One simulation held by the C oracle.  Arrays are numpy float64, shape (nz, ny, nx)
    (x fastest) or flat; materials/fields ``None`` mean the default (see the C file)."""

    FIELD_NAMES = ("Ex", "Ey", "Ez", "Hx", "Hy", "Hz",
                   "Mxx", "Mxy", "Mxz", "Myx", "Myy", "Myz", "Mzx", "Mzy", "Mzz")

    def __init__(self, nx, ny, nz, dx, dy, dz, dt, *, eps_r=None, sigma=None, mu_r=None,
                 Ms=None, alpha=None, gamma=None, bc=(0, 0, 0), enable_llg=True,
                 h_bias=(0.0, 0.0, 0.0), ani_hk=0.0, ani_axis=(0.0, 0.0, 1.0),
                 llg_tol=1e-12, llg_max_iter=20, kind="f64", time_scheme=0, pml=None,
                 pml_r0=1e-6, pml_order=3):
        self._lib, self._p = _lib(kind)
        self.shape = (nz, ny, nx)
        self.n = nx * ny * nz
        f = self._fn("create")
        f.restype = C.c_void_p
        f.argtypes = [C.c_int] * 3 + [C.c_double] * 4 + [_DP] * 6 + [_IP, C.c_int, _DP,
                                                                  C.c_double, _DP, C.c_double,
                                                                  C.c_int]
        mats = [_as_f64(m, self.n) for m in (eps_r, sigma, mu_r, Ms, alpha, gamma)]
        bc_a = (C.c_int * 3)(*[int(b) for b in bc])
        hb = (C.c_double * 3)(*[float(v) for v in h_bias])
        ax = (C.c_double * 3)(*[float(v) for v in ani_axis])
        self._h = f(nx, ny, nz, dx, dy, dz, dt, *[_dptr(m) for m in mats], bc_a,
                    int(bool(enable_llg)), hb, float(ani_hk), ax, float(llg_tol),
                    int(llg_max_iter))
        if not self._h:
            raise ValueError("oracle_create rejected its arguments")
        self._h = C.c_void_p(self._h)
        if time_scheme:   # 1: the first-order scheme of PAPER.md:102-150
            g = self._fn("set_scheme")
            g.restype = C.c_int
            g.argtypes = [C.c_void_p, C.c_int]
            if g(self._h, int(time_scheme)):
                raise ValueError("oracle_set_scheme rejected the scheme")

        if pml is not None and any(int(v) for v in pml):
            # open boundary: pml = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi) cells
            g = self._fn("set_pml")
            g.restype = C.c_int
            g.argtypes = [C.c_void_p, _IP, C.c_double, C.c_int]
            rc = g(self._h, (C.c_int * 6)(*[int(v) for v in pml]), float(pml_r0), int(pml_order))
            if rc:
                raise ValueError(f"oracle_set_pml failed ({rc}): PML on a periodic axis, too thick, "
                                 "or magnetic faces inside the layer")

    def _fn(self, name):
        return getattr(self._lib, self._p + name)

    def set_fields(self, E=(None, None, None), H=(None, None, None), M_cell=(None, None, None)):
        f = self._fn("set_fields")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p] + [_DP] * 9
        arrs = [_as_f64(a, self.n) for a in (*E, *H, *M_cell)]
        rc = f(self._h, *[_dptr(a) for a in arrs])
        if rc:
            raise ValueError(f"oracle_set_fields failed ({rc})")

    def set_source(self, comp, lo, hi, profile=None, amplitude=1.0, f0=0.0, t0=0.0, tp=1.0, kind=0):
        """kind 0 soft E (J of eq. 11), 1 hard E, 2 soft H, 3 hard H (see the C file)."""
        f = self._fn("add_source")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_int, C.c_int, _IP, _IP, _DP] + [C.c_double] * 4
        nb = int(np.prod([h - l for l, h in zip(lo, hi)]))
        prof = _as_f64(profile, nb)
        rc = f(self._h, int(kind), int(comp), (C.c_int * 3)(*lo), (C.c_int * 3)(*hi), _dptr(prof),
               float(amplitude), float(f0), float(t0), float(tp))
        if rc:
            raise ValueError(f"oracle_add_source failed ({rc})")

    def step(self, n=1):
        f = self._fn("step")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_int]
        f(self._h, int(n))

    def hm_half_step(self):
        f = self._fn("hm_half_step")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p]
        f(self._h)

    def read_fields(self, names=None) -> dict:
        names = self.FIELD_NAMES if names is None else names
        out = {nm: np.empty(self.shape, dtype=np.float64) for nm in names}
        ptrs = (_DP * 15)(*[_dptr(out[nm]) if nm in out else None for nm in self.FIELD_NAMES])
        f = self._fn("read_fields")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.POINTER(_DP)]
        f(self._h, ptrs)
        return out

    def write_fields(self, **arrays):
        arrs = {k: _as_f64(v, self.n) for k, v in arrays.items()}
        ptrs = (_DP * 15)(*[_dptr(arrs.get(nm)) for nm in self.FIELD_NAMES])
        f = self._fn("write_fields")
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.POINTER(_DP)]
        f(self._h, ptrs)

    def stats(self) -> dict:
        out = (C.c_double * 8)()
        f = self._fn("get_stats")
        f.argtypes = [C.c_void_p, _DP]
        f(self._h, out)
        keys = ("steps", "time", "iters_last", "iters_max", "iters_total", "nonconverged",
                "resid_last", "halfsteps")
        return dict(zip(keys, list(out)))

    def close(self):
        if getattr(self, "_h", None):
            f = self._fn("destroy")
            f.argtypes = [C.c_void_p]
            f(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def oracle_from_workload(w, kind="f64", time_scheme=0) -> Oracle:
    """An Oracle loaded with a workload description (any object with the attributes of
    ``workloads.Workload``: grid, materials, initial fields, sources, boundary options; its
    ``numpy()`` gives host arrays).  Duck-typed: the oracle imports nothing of the CUDA package."""
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


def omp_threads() -> int:
    """Threads the oracle's OpenMP loops will use (for bench.py's ``cores``)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)
