"""The open boundary (PML, A26) on the CUDA path: parity with the oracle
(<= 1e-9 relative L-inf, as everywhere) with layers on one to six faces, materials running into
the layer, sources inside and outside it, an LLG block in the interior; and the paper's own figure
(< 0.1 % reflection) measured on the GPU result."""
import math

import numpy as np
import pytest
import torch

from tests._util import FIELD_GROUPS, oracle_from_workload, rel_linf
from paper_2103_12819_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-9


def _both(w, steps, **kw):
    from paper_2103_12819_b200.binding import from_workload
    o = oracle_from_workload(w)
    o.step(steps)
    sim = from_workload(w, **kw)
    sim.step(steps)
    return {k: v.numpy() for k, v in sim.read_fields().items()}, o.read_fields(), sim, o


@pytest.mark.parametrize("pml", [(6, 6, 0, 0, 0, 0), (5, 0, 0, 7, 4, 6), (8, 8, 8, 8, 8, 8)])
def test_maxwell_with_materials_and_sources_in_a_pml_box(pml):
    """config-3-like: dielectric slab and conductor strips run INTO the layer (PAPER.md:189:
    "material aligned with the domain boundaries"); the soft source plane crosses it too."""
    w = wl.make_config(3, shape=(72, 40, 36))
    w.pml = pml
    got, ref, sim, _ = _both(w, 120)
    for g in ("E", "H"):
        assert rel_linf(got, ref, g) <= TOL, (g, rel_linf(got, ref, g))
    assert max(np.abs(ref[n]).max() for n in FIELD_GROUPS["E"]) > 0
    # chunked plain launches == one graph replay
    from paper_2103_12819_b200.binding import from_workload
    alt = from_workload(w, use_graph=False)
    for c in (1, 2, 117):
        alt.step(c)
    alt = {k: v.numpy() for k, v in alt.read_fields().items()}
    for n in FIELD_GROUPS["E"] + FIELD_GROUPS["H"]:
        assert np.array_equal(got[n], alt[n]), n


@pytest.mark.parametrize("kernel_path", [5, 1])
def test_llg_block_inside_a_box_open_on_five_sides(kernel_path):
    """A magnetic block (config 4's material, anisotropy, bias) in the middle of a box whose x, y
    and upper z faces are open; hard and soft sources outside the layer."""
    w = wl.make_config(4, shape=(44, 36, 40))
    Ms = w.materials["Ms"]
    blk = torch.zeros_like(Ms)
    blk[12:28, 10:26, 12:32] = 1.4e5
    w.materials["Ms"] = blk
    w.M_cell = wl.tilted_m_cell(w.seed, w.nx, w.ny, w.nz, blk, 0.5, "cpu")
    w.pml = (6, 6, 5, 5, 0, 7)
    w.sources = [wl.Source(0, (10, 8, 9), (34, 28, 10), 1e12, 5e12, 30 * w.dt, 20 * w.dt, None, 0),
                 wl.Source(1, (20, 6, 20), (21, 30, 21), 5e5, 5e12, 30 * w.dt, 20 * w.dt, None, 1)]
    got, ref, sim, o = _both(w, 100, kernel_path=kernel_path)
    for g in ("E", "H", "M"):
        assert rel_linf(got, ref, g) <= TOL, (g, rel_linf(got, ref, g))
    assert sim.stats()["iters_total"] == int(o.stats()["iters_total"]) > 0
    assert float(np.abs(got["Mxy"]).max()) > 0


def test_reflection_below_a_tenth_of_a_percent_on_the_gpu():
    """PAPER.md:189, measured on the CUDA result: a pulse sent into a 12-cell layer of a vacuum
    column; the same column without the layer sends everything back."""
    from paper_2103_12819_b200.binding import FdtdLlg
    nx, pml, dx = 300, 12, 1e-3
    c0 = 299792458.0
    dt = 0.5 * dx / c0
    i = np.arange(nx)
    ey = np.exp(-0.5 * ((i - 0.35 * nx) / 8.0) ** 2).reshape(1, 1, nx)
    hz = (np.exp(-0.5 * ((i + 0.5 - 0.35 * nx) / 8.0) ** 2) / (4e-7 * math.pi * c0)).reshape(1, 1, nx)
    steps = int(((nx - pml - 0.35 * nx) + 0.45 * nx) * dx / (c0 * dt))
    out = {}
    for name, p in (("open", (pml, pml, 0, 0, 0, 0)), ("wall", None)):
        sim = FdtdLlg(nx, 1, 1, dx, dx, dx, dt, bc=(0, 1, 1), enable_llg=False, pml=p)
        sim.set_fields([None, torch.from_numpy(ey), None], [None, None, torch.from_numpy(hz)], None)
        sim.step(steps)
        out[name] = sim.read_fields(names=("Ey",))["Ey"].numpy()[0, 0]
    assert np.max(np.abs(out["wall"])) > 0.9
    assert np.max(np.abs(out["open"][pml:nx - pml])) < 1e-3


def test_pml_argument_errors():
    from paper_2103_12819_b200.binding import FdtdLlg, FdtdLlgError
    with pytest.raises(FdtdLlgError):      # periodic axis
        FdtdLlg(8, 8, 8, 1e-3, 1e-3, 1e-3, 1e-12, bc=(1, 0, 0), enable_llg=False, pml=(2, 0, 0, 0, 0, 0))
    with pytest.raises(FdtdLlgError):      # magnetic cells in the layer
        FdtdLlg(8, 8, 8, 1e-3, 1e-3, 1e-3, 1e-12, bc=(0, 0, 0), enable_llg=True,
                materials={"Ms": 1e5, "alpha": 0.1, "gamma": 1.7e11}, pml=(2, 0, 0, 0, 0, 0))
    sim = FdtdLlg(8, 8, 8, 1e-3, 1e-3, 1e-3, 1e-12, bc=(0, 0, 0), enable_llg=False, pml=(2, 2, 0, 0, 0, 0))
    with pytest.raises(FdtdLlgError):      # hard source inside the layer
        sim.set_source(1, (0, 0, 0), (3, 8, 8), None, 1.0, 0.0, 0.0, 1e-12, kind=1)
