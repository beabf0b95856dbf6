"""z-slab decomposition (fdtd_llg.h "Z-SLABS") on ONE GPU.

Several slab handles of one grid live on the same device and hand their boundary planes to each
other with the same peer stores the multi-GPU run uses (the "peer" workspace is local).  Every
update is a Jacobi sweep, so the slabs must hold, BIT FOR BIT, what one handle on the whole grid
holds -- fields, iteration counts -- whatever the cut does to magnetic interfaces, source planes,
periodic axes or the kernel path.  A second test runs the slabs in two PROCESSES that map each
other's workspace with CUDA IPC (gloo carries the 8-byte residual word through the host: no kernel
ever waits on another, so sharing one GPU is safe); NCCL replaces gloo on a multi-GPU node.
"""
import os
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest
import torch

from tests._util import FIELD_GROUPS
from paper_2103_12819_b200 import workloads as wl

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent
ALL = FIELD_GROUPS["E"] + FIELD_GROUPS["H"] + FIELD_GROUPS["M"]


def _single(w, steps, **kw):
    from paper_2103_12819_b200.binding import from_workload
    sim = from_workload(w, **kw)
    sim.step(steps)
    return {k: v.numpy() for k, v in sim.read_fields().items()}, sim.stats()


def _everything(bc, shape=(37, 11, 12)):
    """Spatially varying everything (the workload of test_parity_gpu's boundary-mix test)."""
    rng = np.random.default_rng(11)
    nx, ny, nz = shape
    shp = (nz, ny, nx)
    w = wl.Workload("everything", nx, ny, nz, 1e-6, 1.2e-6, 0.8e-6,
                    wl.courant_dt(0.9, 1e-6, 1.2e-6, 0.8e-6), bc, 30, enable_llg=True,
                    h_bias=(1e3, -2e3, 1e4), ani_hk=3e3, ani_axis=(0.6, 0.0, 0.8),
                    llg_tol=1e-13, llg_max_iter=30)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    Ms = 1.4e5 * (1 + rng.random(shp)) * (rng.random(shp) < 0.6)
    Ms[:, :, 30:] = 0.0
    mu = np.where(Ms > 0, 1.0, 1 + rng.random(shp) * (rng.random(shp) < 0.3))
    w.materials = {"eps_r": t(1 + 3 * rng.random(shp)),
                   "sigma": t(100 * rng.random(shp) * (rng.random(shp) < 0.5)),
                   "mu_r": t(mu), "Ms": t(Ms), "alpha": t(0.01 + 0.05 * rng.random(shp)),
                   "gamma": t(-1.759e11 * (1 + 0.1 * rng.random(shp)))}
    th, ph = np.pi * rng.random(shp), 2 * np.pi * rng.random(shp)
    w.M_cell = [t(Ms * np.sin(th) * np.cos(ph)), t(Ms * np.sin(th) * np.sin(ph)), t(Ms * np.cos(th))]
    w.E = [t(1e6 * rng.standard_normal(shp)) for _ in range(3)]
    w.H = [t(1e3 * rng.standard_normal(shp)) for _ in range(3)]
    lo, hi = (1, 2, 1), (nx - 1, 5, 7)          # spans several slabs
    nb = [h - l for l, h in zip(lo, hi)]
    w.sources = [wl.Source(1, lo, hi, 1e12, 2e12, 3e-15, 2e-15, profile=t(rng.random((nb[2], nb[1], nb[0])))),
                 wl.Source(2, (0, 0, 0), shape, 5e11, 1e12, 1e-15, 4e-15),
                 wl.Source(0, (3, 0, 5), (20, ny, 7), 4e5, 1e12, 1e-15, 4e-15, kind=1)]   # hard E across a cut
    return w


CASES = [
    # (config, shape, slabs, kernel_path, merge_h)
    (5, (40, 44, 36), 2, 0, True),     # the cut IS the magnetic interface (k = 18); periodic x, y
    (5, (40, 44, 36), 3, 5, True),     # interface inside slab 1; staged sweeps forced
    (5, (40, 44, 36), 4, 1, False),    # two half-steps everywhere
    (4, (44, 36, 40), 2, 0, True),     # PEC box, anisotropy, soft source; the cut is in vacuum
    (4, (44, 36, 40), 10, 0, True),    # 4 planes per slab: the slab top (k = 3) + halo straddle a cut, source plane k = 5 in slab 1
    (1, (32, 32, 32), 4, 5, True),     # every cell magnetic: uniform maps, every cut inside the magnet
    (2, (40, 36, 28), 4, 0, True),     # Maxwell only, PERIODIC z closed over the end slabs
    (2, (40, 36, 28), 2, 0, False),
    (5, (24, 20, 6), 6, 0, True),      # one plane per slab: every plane is first and last
]


@pytest.mark.parametrize("cfg,shape,world,path,merge", CASES)
def test_slabs_hold_what_one_handle_holds_bit_for_bit(cfg, shape, world, path, merge):
    from paper_2103_12819_b200.slabs import LocalSlabs
    w = wl.make_config(cfg, shape=shape)
    steps = 12
    ref, st = _single(w, steps, kernel_path=path, merge_h=merge)
    grp = LocalSlabs(w, world, kernel_path=path, merge_h=merge)
    grp.step(steps)
    got = grp.read_fields()
    for n in ALL:
        assert np.array_equal(got[n], ref[n]), (n, float(np.max(np.abs(got[n] - ref[n]))))
    if w.enable_llg:
        its = [s.stats() for s in grp.sims]
        mag = [s for s in its if s["sweep_cells"] > 0]
        assert mag and all(s["iters_total"] == st["iters_total"] for s in mag)
        assert all(s["nonconverged_halfsteps"] == 0 for s in its)
        assert sum(s["magnetic_cells"] for s in its) == st["magnetic_cells"]
        # the host looked at the residual once per half-step, not once per iterate
        assert grp.host_checks <= 2 * steps * max(1, (st["iters_max"] + 2) // 3)
    assert max(float(np.max(np.abs(ref[n]))) for n in FIELD_GROUPS["H"]) > 0


def test_iteration_count_falls_again_with_slabs_that_hold_no_magnet():
    """Config 4 on 24 x 20 x 40 at tol 1e-10: the pulse takes the iteration count from 2 to 3 and back
    (the oracle's history of this workload), and three of the four slabs have no magnetic face.  Their
    residual words receive the maximum over all slabs with every merge; unless the closing sub-step
    clears them there too, the stopping test turns into a running maximum over the
    past and the count never comes down again."""
    from paper_2103_12819_b200.slabs import LocalSlabs
    w = wl.make_config(4, shape=(24, 20, 40))
    w.llg_tol = 1e-10
    steps = 40
    ref, st = _single(w, steps)
    assert st["iters_max"] == 3 and 2 * 2 * steps < st["iters_total"] < 3 * 2 * steps   # 2, then 3, then 2
    assert st["iters_last"] == 2
    grp = LocalSlabs(w, 4)
    its = [s.stats() for s in grp.sims]
    assert [s["sweep_cells"] > 0 for s in its] == [True, False, False, False]
    grp.step(steps)
    got = grp.read_fields()
    its = [s.stats() for s in grp.sims]
    assert its[0]["iters_total"] == st["iters_total"] and its[0]["iters_last"] == 2
    assert all(s["nonconverged_halfsteps"] == 0 for s in its)
    for n in ALL:
        assert np.array_equal(got[n], ref[n]), (n, float(np.max(np.abs(got[n] - ref[n]))))


@pytest.mark.parametrize("bc", [(1, 0, 1), (0, 1, 0), (1, 1, 1)])
def test_slabs_with_every_material_array_and_sources_across_the_cuts(bc):
    from paper_2103_12819_b200.slabs import LocalSlabs
    w = _everything(bc)
    ref, st = _single(w, 20)
    for world in (3, 4):
        grp = LocalSlabs(w, world)
        grp.step(20)
        got = grp.read_fields()
        for n in ALL:
            assert np.array_equal(got[n], ref[n]), (world, n)
        assert all(s.stats()["iters_total"] == st["iters_total"] for s in grp.sims if s.stats()["sweep_cells"])


def test_substeps_on_a_plain_handle_equal_step():
    """fdtd_llg_substep on a handle without interfaces: the same kernels in the same order."""
    from paper_2103_12819_b200.slabs import LocalSlabs
    for cfg in (4, 3):
        w = wl.make_config(cfg, shape=wl.SMALL_SHAPES[cfg])
        ref, st = _single(w, 15)
        grp = LocalSlabs(w, 1)
        grp.step(15)
        got = grp.read_fields()
        for n in ALL:
            assert np.array_equal(got[n], ref[n]), n
        assert grp.sims[0].stats()["steps"] == 15


def test_out_of_order_substeps_and_step_on_a_connected_slab_are_refused():
    from paper_2103_12819_b200 import binding as B
    from paper_2103_12819_b200.slabs import LocalSlabs
    w = wl.make_config(5, shape=(24, 20, 8))
    grp = LocalSlabs(w, 2)
    a = grp.sims[0]
    with pytest.raises(B.FdtdLlgError) as e:
        a.step(1)
    assert e.value.code == B.ESTATE
    with pytest.raises(B.FdtdLlgError) as e:
        a.substep(B.SUB_E)
    assert e.value.code == B.ESTATE
    a.substep(B.SUB_BEGIN)
    with pytest.raises(B.FdtdLlgError):
        a.substep(B.SUB_HM1, 2)            # iterate 2 before iterate 1
    with pytest.raises(B.FdtdLlgError):
        a.read_fields()                    # a step is open
    # shapes must agree
    other = B.from_workload(wl.make_config(5, shape=(24, 20, 6)), use_graph=False)
    with pytest.raises(B.FdtdLlgError) as e:
        grp.sims[1].connect((other.slab_info(), other.workspace.data_ptr()), None)
    assert e.value.code in (B.EINVAL, B.ESTATE)
    # merge_h is a property of the whole grid: slabs that disagree are refused, and so is an H source
    # (which switches it off) on a connected slab
    from paper_2103_12819_b200.slabs import cut_workload, plan_slabs
    plans = plan_slabs(w.nz, 2, False)
    lo = B.from_workload(cut_workload(w, plans[0]), use_graph=False, merge_h=True)
    hi = B.from_workload(cut_workload(w, plans[1]), use_graph=False, merge_h=False)
    with pytest.raises(B.FdtdLlgError) as e:
        lo.connect(None, (hi.slab_info(), hi.workspace.data_ptr()))
    assert e.value.code == B.EINVAL and "merge_h" in str(e.value)
    grp2 = LocalSlabs(w, 2)
    with pytest.raises(B.FdtdLlgError) as e:
        grp2.sims[0].set_source(0, (0, 0, 0), (4, 4, 2), kind=3)
    assert e.value.code == B.ESTATE and "merge_h" in str(e.value)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("cfg,shape", [(5, (40, 44, 36)), (2, (40, 36, 28)), (4, (44, 36, 40))])
def test_two_processes_map_each_other_with_cuda_ipc(cfg, shape, tmp_path):
    """One process per slab (as on a multi-GPU node), here both on GPU 0: workspaces exchanged as
    CUDA IPC handles, boundary planes stored straight into the other process's ghost planes."""
    steps = 10
    w = wl.make_config(cfg, shape=shape)
    ref, st = _single(w, steps)
    port = _free_port()
    outs = [tmp_path / f"slab{r}.npz" for r in range(2)]
    procs = [subprocess.Popen([sys.executable, str(ROOT / "tests" / "slab_worker.py"), str(r), "2", str(port),
                               str(cfg), ",".join(map(str, shape)), str(steps), str(outs[r])],
                              cwd=str(ROOT), env=dict(os.environ, PYTHONPATH=str(ROOT)))
             for r in range(2)]
    for p in procs:
        assert p.wait(timeout=600) == 0
    parts = [np.load(o) for o in outs]
    for n in ALL:
        got = np.concatenate([p[n] for p in parts], 0)
        assert np.array_equal(got, ref[n]), n
    if w.enable_llg:
        assert int(parts[0]["iters_total"]) == st["iters_total"]


def test_slabs_first_order_scheme_and_open_boundary_with_hard_h_source():
    """The other step variants across cuts: the first-order scheme (one explicit sweep per half-step),
    and the paper's tunable-filter set-up in small (PML at the z-low end, hard H source on the last
    plane, LLG slab on a side wall, dielectric array: the H half-steps are merged outside the margins
    -- the layer, the source plane -- and k_pml runs on the end slab only)."""
    from paper_2103_12819_b200.slabs import LocalSlabs
    w = wl.make_config(5, shape=(40, 44, 36))
    ref, st = _single(w, 10, time_scheme=1)
    grp = LocalSlabs(w, 3, time_scheme=1)
    grp.step(10)
    got = grp.read_fields()
    for n in ALL:
        assert np.array_equal(got[n], ref[n]), n
    w = wl.paper_tunable_filter(nx=96, ny=4, nz=48, npml=8)
    ref, st = _single(w, 40)
    assert st["merged_h"] == 1      # merged outside the margins: the PML layer and the source plane
    for world in (2, 3):
        grp = LocalSlabs(w, world)
        grp.step(40)
        got = grp.read_fields()
        for n in ALL:
            assert np.array_equal(got[n], ref[n]), (world, n)
    assert max(float(np.max(np.abs(ref[n]))) for n in FIELD_GROUPS["M"]) > 0
