"""Parity of the CUDA path (through the C ABI) against the CPU oracle -- the first gate.

Same seeded inputs on both sides; element-by-element comparison; the bar is BASELINE.json's:
max relative L-infinity error <= 1e-9 on E, H and M after 100 steps (A21 defines the
norm).  Shapes span several 32x4x2 thread blocks plus a ragged tail in every axis.
"""
import numpy as np
import pytest
import torch

from tests._util import FIELD_GROUPS, oracle_from_workload, record_parity, rel_linf, rel_linf_of_change
from paper_2103_12819_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-9  # north_star: max relative L-inf on E, H and M after 100 steps


def _gpu_fields(sim):
    return {k: v.numpy() for k, v in sim.read_fields().items()}


def _run_both(w, steps, use_graph=True, chunks=(None,)):
    from paper_2103_12819_b200.binding import from_workload
    o = oracle_from_workload(w)
    o.step(steps)
    ref = o.read_fields()
    sim = from_workload(w, use_graph=use_graph)
    if chunks == (None,):
        sim.step(steps)
    else:
        for c in chunks:
            sim.step(c)
    got = _gpu_fields(sim)
    return got, ref, sim.stats(), o.stats()


def _assert_parity(got, ref, llg, tol=TOL, record=None):
    errs = {g: rel_linf(got, ref, g) for g in ("E", "H") + (("M",) if llg else ())}
    if record is not None:
        record_parity(dict(record, **{"err_" + g: e for g, e in errs.items()}))
    for g, e in errs.items():
        assert e <= tol, (g, errs)
    return errs


def _assert_m_error_small_against_its_change(got, ref, w, tol=1e-6, **oracle_kw):
    """|M| = Ms never moves, so an error of 1e-9 Ms says little about a run in which M turns by a
    fraction of a radian: measure the error against how far M moved (a wrong damping or anisotropy
    term shows here first)."""
    ref0 = oracle_from_workload(w, **oracle_kw).read_fields()
    assert max(float(np.max(np.abs(ref[n] - ref0[n]))) for n in FIELD_GROUPS["M"]) > 0   # M moved
    e = rel_linf_of_change(got, ref, ref0, "M")
    assert e <= tol, e
    return e


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_parity_100_steps_all_configs(cfg):
    """On these shapes the default kernel_path picks the direct-load sweeps (the box is too small
    to give every SM an item); the staged sweeps are forced with kernel_path 5 below and run by
    default at the sizes of test_fullsize_gpu.py and of the every-SM-busy test."""
    w = wl.make_config(cfg, shape=wl.SMALL_SHAPES[cfg])
    got, ref, gs, os_ = _run_both(w, 100)
    from paper_2103_12819_b200.binding import from_workload
    sim = from_workload(w, kernel_path=5)     # staged LLG sweeps and staged / fused Maxwell sweeps forced
    if w.enable_llg:
        assert sim.stats()["staged_sweeps"] == 1 and gs["staged_sweeps"] == 0
    sim.step(100)
    _assert_parity(_gpu_fields(sim), ref, w.enable_llg,
                   record={"test": "parity_100_steps_small", "config": cfg, "shape": list(wl.SMALL_SHAPES[cfg]),
                           "steps": 100, "path": "staged (kernel_path 5)"})
    _assert_parity(got, ref, w.enable_llg,
                   record={"test": "parity_100_steps_small", "config": cfg, "shape": list(wl.SMALL_SHAPES[cfg]),
                           "steps": 100, "path": "default", "iters": gs["iters_total"]})
    assert gs["steps"] == 100
    if w.enable_llg:
        # same number of LLG iterations, all converged
        assert gs["iters_total"] == int(os_["iters_total"])
        assert gs["nonconverged_halfsteps"] == 0
        assert gs["halfsteps"] == 200
        _assert_m_error_small_against_its_change(got, ref, w)
        _assert_m_error_small_against_its_change(_gpu_fields(sim), ref, w)
        # wall faces / non-magnetic faces carry exactly M = 0 on both sides
        for n in FIELD_GROUPS["M"]:
            assert np.array_equal(got[n] == 0.0, ref[n] == 0.0)
    # the fields are not trivially zero
    assert max(np.abs(ref[n]).max() for n in FIELD_GROUPS["E"]) > 0


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1), (1, 0, 1), (0, 1, 1), (1, 1, 0)])
def test_parity_every_boundary_mix_with_everything_on(bc):
    """Spatially varying eps, sigma, mu, Ms, alpha, gamma, anisotropy, two sources with and
    without profile, partially magnetic box: all template branches of the kernels."""
    rng = np.random.default_rng(5)
    shape = (37, 11, 9)
    nx, ny, nz = shape
    shp = (nz, ny, nx)
    w = wl.Workload("everything", nx, ny, nz, 1e-6, 1.2e-6, 0.8e-6,
                    wl.courant_dt(0.9, 1e-6, 1.2e-6, 0.8e-6), bc, 30, enable_llg=True,
                    h_bias=(1e3, -2e3, 1e4), ani_hk=3e3, ani_axis=(0.6, 0.0, 0.8),
                    llg_tol=1e-13, llg_max_iter=30)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    Ms = 1.4e5 * (1 + rng.random(shp)) * (rng.random(shp) < 0.6)
    Ms[:, :, 30:] = 0.0          # the sweep box does not cover the whole grid
    mu = np.where(Ms > 0, 1.0, 1 + rng.random(shp) * (rng.random(shp) < 0.3))
    w.materials = {"eps_r": t(1 + 3 * rng.random(shp)),
                   "sigma": t(100 * rng.random(shp) * (rng.random(shp) < 0.5)),
                   "mu_r": t(mu), "Ms": t(Ms), "alpha": t(0.01 + 0.05 * rng.random(shp)),
                   "gamma": t(-1.759e11 * (1 + 0.1 * rng.random(shp)))}
    th, ph = np.pi * rng.random(shp), 2 * np.pi * rng.random(shp)
    w.M_cell = [t(Ms * np.sin(th) * np.cos(ph)), t(Ms * np.sin(th) * np.sin(ph)), t(Ms * np.cos(th))]
    w.E = [t(1e6 * rng.standard_normal(shp)) for _ in range(3)]
    w.H = [t(1e3 * rng.standard_normal(shp)) for _ in range(3)]
    lo, hi = (1, 2, 1), (nx - 1, 5, 4)
    nb = int(np.prod([h - l for l, h in zip(lo, hi)]))
    w.sources = [wl.Source(1, lo, hi, 1e12, 2e12, 3e-15, 2e-15, profile=t(rng.random(nb))),
                 wl.Source(2, (0, 0, 0), shape, 5e11, 1e12, 1e-15, 4e-15)]
    got, ref, gs, os_ = _run_both(w, 30)
    _assert_parity(got, ref, True)
    assert gs["iters_total"] == int(os_["iters_total"])


def test_graph_and_plain_launches_agree_bitwise_and_step_chunks():
    """step(100) == step(37)+step(63) == the same without a CUDA graph, bit for bit."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(4, shape=wl.SMALL_SHAPES[4])
    outs = []
    for use_graph, chunks in ((True, (100,)), (True, (37, 63)), (False, (100,))):
        sim = from_workload(w, use_graph=use_graph)
        for c in chunks:
            sim.step(c)
        outs.append(_gpu_fields(sim))
        assert sim.stats()["steps"] == 100
        st = sim.stats()
        # + the launches that take the merged faces to t = dt/2 before the first step (<= 6 slabs)
        assert 0 <= st["kernel_launches"] - 100 * st["launches_per_step"] <= 6
    for other in outs[1:]:
        for n in outs[0]:
            assert np.array_equal(outs[0][n], other[n]), n


@pytest.mark.parametrize("cfg,shape", [(1, (32, 32, 32)), (4, (44, 36, 40)), (5, (40, 44, 36)),
                                       (5, (70, 19, 23)), (4, (33, 8, 50))])
def test_staged_and_tma_sweeps_equal_direct_load_kernels_bitwise(cfg, shape):
    """kernel_path 5 (staged sweeps: TMA-fed shared-memory ring, thread = cell) and 1 (direct
    global loads) share the arithmetic (hm_face_core): every field and the iteration counts agree
    bit for bit, on shapes with ragged tiles in x and y and several z chunks."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(cfg, shape=shape)
    outs, stats = [], []
    for path in (1, 5):
        sim = from_workload(w, kernel_path=path)
        assert sim.stats()["staged_sweeps"] == (path != 1)
        sim.step(25)
        outs.append(_gpu_fields(sim))
        stats.append(sim.stats())
    for n in outs[0]:
        assert np.array_equal(outs[0][n], outs[1][n]), n
    assert stats[0]["iters_total"] == stats[1]["iters_total"] > 0


@pytest.mark.parametrize("cfg,shape", [(2, (40, 36, 28)), (3, (72, 40, 36)), (3, (70, 33, 50)), (4, (44, 36, 40)),
                                       (5, (70, 19, 23)), (2, (33, 17, 40))])
def test_fused_maxwell_sweep_equals_the_separate_kernels_bitwise(cfg, shape):
    """kernel_path 5 forces the staged sweeps of eh_stage.cuh (eq. 11 from a TMA-fed ring, fused with
    the merged H update outside the LLG box); kernel_path 1 runs k_e_update + k_h_update with direct
    loads.  They share e_edge_val / h_face_val: the same bits, on ragged tiles, with material
    arrays (config 3), a soft source, periodic and PEC ends."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(cfg, shape=shape)
    outs = []
    for path in (1, 5):
        sim = from_workload(w, kernel_path=path)
        assert sim.stats()["merged_h"] == 1
        sim.step(30)
        outs.append(_gpu_fields(sim))
    for n in outs[0]:
        assert np.array_equal(outs[0][n], outs[1][n]), (n, float(np.max(np.abs(outs[0][n] - outs[1][n]))))


@pytest.mark.parametrize("cfg,shape", [(2, (40, 36, 28)), (2, (33, 31, 26)), (5, (40, 44, 36)), (5, (70, 19, 23))])
def test_fused_sweep_carries_the_soft_current_onto_the_periodic_image(cfg, shape):
    """A soft E source whose box touches index 0 of a periodic axis: the fused sweep recomputes
    E^{n+1} at index n (the image of index 0) on the rim of its last tiles and must put
    the same J there (eq. 11), or H at n-1 is built from an E without the current.
    kernel_path 1 reads the stored ghost image instead: both must give the same bits, and the
    oracle's values to 1e-9."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(cfg, shape=shape)
    nx, ny, nz = shape
    rng = np.random.default_rng(5)
    f0, t0, tp = 3.0 / (40 * w.dt), 12 * w.dt, 5 * w.dt

    def box_source(comp, lo, hi, amp):
        nb = int(np.prod([h - l for l, h in zip(lo, hi)]))
        return wl.Source(comp, lo, hi, amp, f0, t0, tp, profile=torch.from_numpy(0.5 + rng.random(nb)))

    w.sources = list(w.sources) + [
        box_source(0, (3, 0, 0), (nx - 2, 2, 3), 4e10),          # J_x from index 0 in y and z
        box_source(1, (0, 2, 0), (3, ny - 1, 2), 3e10),          # J_y from index 0 in x and z
        box_source(2, (0, 0, 1), (2, 3, nz - 1), 5e10),          # J_z from index 0 in x and y
        wl.Source(2, (0, 0, 0), shape, 1e10, f0, t0, tp),        # everywhere, no profile
    ]
    outs = []
    for path in (1, 5):
        sim = from_workload(w, kernel_path=path)
        st = sim.stats()
        assert st["merged_h"] == 1
        if path == 5:   # the fused sweep runs: everywhere (config 2) / outside the LLG box (config 5)
            assert st["staged_maxwell"] == 2
        sim.step(30)
        outs.append(_gpu_fields(sim))
    for n in outs[0]:
        assert np.array_equal(outs[0][n], outs[1][n]), (n, float(np.max(np.abs(outs[0][n] - outs[1][n]))))
    o = oracle_from_workload(w)
    o.step(30)
    _assert_parity(outs[1], o.read_fields(), w.enable_llg)


def test_merged_h_equals_two_half_steps_to_rounding_and_reads_do_not_disturb():
    """merge_h: one update instead of two half-steps with the same curl E: equal up to rounding
    (1 ulp per step), and reading the fields mid-run (which forms the integer-time H) changes nothing."""
    from paper_2103_12819_b200.binding import from_workload
    for cfg in (3, 4):
        w = wl.make_config(cfg, shape=wl.SMALL_SHAPES[cfg])
        a = from_workload(w, merge_h=False)
        b = from_workload(w, merge_h=True)
        c = from_workload(w, merge_h=True)
        assert a.stats()["merged_h"] == 0 and b.stats()["merged_h"] == 1
        a.step(60)
        b.step(60)
        for n in (7, 1, 22, 30):
            c.step(n)
            mid = _gpu_fields(c)
            again = _gpu_fields(c)          # a second read of the same state
            for k in mid:
                assert np.array_equal(mid[k], again[k]), k
        fa, fb, fc = _gpu_fields(a), _gpu_fields(b), _gpu_fields(c)
        for k in fb:
            assert np.array_equal(fb[k], fc[k]), k
        for g_ in ("E", "H") + (("M",) if w.enable_llg else ()):
            assert rel_linf(fb, fa, g_) < 1e-13, (cfg, g_, rel_linf(fb, fa, g_))


@pytest.mark.parametrize("cfg,shape", [(5, (200, 176, 300)), (4, (230, 150, 200))])
def test_kernel_paths_agree_bitwise_with_every_sm_busy(cfg, shape):
    """The staged sweeps hand out work items dynamically and stream through mbarrier rings; with
    thousands of items in flight on all SMs a producer / consumer race or a stale stage would
    change bits.  Jacobi sweeps are order independent, so every path and every repetition must
    give the same bits as the direct-load kernels."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(cfg, shape=shape, device="cuda:0")
    ref = None
    for path in (1, 0, 0, 5):
        sim = from_workload(w, kernel_path=path)
        sim.step(4)
        got = {k: v for k, v in sim.read_fields(device="cuda:0").items()}
        assert sim.stats()["nonconverged_halfsteps"] == 0
        if ref is None:
            ref = got
            continue
        for n in ref:
            assert torch.equal(ref[n], got[n]), (path, n)
        del got, sim


@pytest.mark.parametrize("tol,iters", [(1e-2, 1), (1e-7, 2)])
def test_early_stop_after_one_or_two_iterates_on_every_kernel_path(tol, iters):
    """A loose tolerance stops the iteration at R = 1 or at R = 2 (even R: the result sits in the
    pong H set and is copied to the canonical one)."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(5, shape=(40, 44, 36))
    w.llg_tol = tol
    o = oracle_from_workload(w)
    o.step(20)
    ref = o.read_fields()
    assert int(o.stats()["iters_total"]) == 40 * iters
    outs = []
    for path in (1, 5):
        sim = from_workload(w, kernel_path=path)
        sim.step(20)
        outs.append(_gpu_fields(sim))
        assert sim.stats()["iters_total"] == 40 * iters and sim.stats()["iters_max"] == iters
    for got in outs:
        _assert_parity(got, ref, True)
    for n in outs[0]:
        assert np.array_equal(outs[0][n], outs[1][n]), n


@pytest.mark.parametrize("cfg", [1, 4, 5])
def test_first_order_scheme_parity_100_steps(cfg):
    """time_scheme = 1: one forward-Euler sweep per (H,M) half-step.  Same bar
    as the second-order scheme; every kernel path agrees bit for bit."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(cfg, shape=wl.SMALL_SHAPES[cfg])
    o = oracle_from_workload(w, time_scheme=1)
    o.step(100)
    ref = o.read_fields()
    outs = []
    for path in (5, 1):
        sim = from_workload(w, kernel_path=path, time_scheme=1)
        sim.step(100)
        outs.append(_gpu_fields(sim))
        st = sim.stats()
        assert st["iters_total"] == int(o.stats()["iters_total"]) == 200   # one sweep per half-step
        assert st["nonconverged_halfsteps"] == 0
    _assert_parity(outs[0], ref, True)
    _assert_m_error_small_against_its_change(outs[0], ref, w, time_scheme=1)
    for other in outs[1:]:
        for n in outs[0]:
            assert np.array_equal(outs[0][n], other[n]), n
    # and it is not the second-order result
    o2 = oracle_from_workload(w)
    o2.step(100)
    assert rel_linf(o2.read_fields(), ref, "M") > 1e-9


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1), (1, 0, 1)])
def test_hard_and_soft_field_sources(bc):
    """All four source kinds of fdtd_llg_add_source on a config-4-like grid (magnetic
    slab, anisotropy), boxes cut by walls and by periodic ends; 60 steps, graph replay."""
    from paper_2103_12819_b200.binding import from_workload
    w = wl.make_config(4, shape=(44, 36, 40))
    w.bc = bc
    g = torch.Generator().manual_seed(7)
    f0, tp, t0 = 5e12, 20 * w.dt, 30 * w.dt
    w.sources = []
    for kind, comp, lo, hi, A in ((0, 0, (0, 0, 4), (44, 36, 5), 1e12), (1, 1, (0, 0, 0), (9, 36, 7), 5e5),
                                  (2, 2, (40, 0, 0), (44, 36, 40), 3e16), (3, 0, (0, 30, 0), (3, 36, 40), 2e2),
                                  (1, 2, (20, 20, 2), (21, 21, 38), -1e6), (3, 1, (5, 0, 0), (40, 1, 6), 1e2)):
        nb = [h - l for l, h in zip(lo, hi)]
        prof = torch.rand((nb[2], nb[1], nb[0]), generator=g, dtype=torch.float64)
        w.sources.append(wl.Source(comp, lo, hi, A, f0, t0, tp, prof, kind))
    got, ref, gs, os_ = _run_both(w, 60)
    _assert_parity(got, ref, True)
    assert gs["iters_total"] == int(os_["iters_total"])
    # the sources dominate the fields: a run without them is different
    w2 = wl.make_config(4, shape=(44, 36, 40))
    w2.bc = bc
    w2.sources = []
    o = oracle_from_workload(w2)
    o.step(60)
    assert rel_linf(o.read_fields(), ref, "E") > 1e-2
    # chunked stepping and plain launches give the same bits as one graph replay of 60 steps
    sim = from_workload(w, use_graph=False)
    for c in (1, 2, 57):
        sim.step(c)
    alt = _gpu_fields(sim)
    for n in got:
        assert np.array_equal(got[n], alt[n]), n


def test_device_resident_inputs_equal_host_inputs():
    from paper_2103_12819_b200.binding import from_workload
    wh = wl.make_config(5, shape=wl.SMALL_SHAPES[5])
    wd = wl.make_config(5, shape=wl.SMALL_SHAPES[5], device="cuda:0")
    # the generator is counter based: host and device give the same inputs (to libm rounding)
    for a, b in zip(wh.E + wh.M_cell, wd.E + wd.M_cell):
        assert torch.allclose(a, b.cpu(), rtol=1e-13, atol=1e-13 * float(a.abs().max()))
    sh, sd = from_workload(wh), from_workload(wd)
    sh.step(20)
    sd.step(20)
    fh, fd = _gpu_fields(sh), {k: v.cpu().numpy() for k, v in sd.read_fields(device="cuda:0").items()}
    for g in ("E", "H", "M"):
        assert rel_linf(fd, fh, g) < 1e-11


@pytest.mark.parametrize("shape,bc", [((1, 1, 1), (1, 1, 1)), ((1, 5, 3), (1, 0, 1)),
                                      ((2, 2, 2), (0, 0, 0)), ((33, 1, 2), (1, 1, 0)),
                                      ((64, 8, 4), (1, 1, 1)), ((65, 9, 5), (0, 0, 0))])
def test_degenerate_and_ragged_shapes(shape, bc):
    """Single-cell axes (periodic neighbours are the cell itself), grids smaller than one thread
    block, exact multiples of the block and one more."""
    w = wl.config5(shape=shape)
    w.bc = bc
    got, ref, gs, os_ = _run_both(w, 12)
    _assert_parity(got, ref, True)
    assert gs["iters_total"] == int(os_["iters_total"])


def test_iteration_cap_is_accepted_and_counted():
    """A4: at llg_max_iter the iterate is accepted and the half-step counted as non-converged."""
    w = wl.make_config(1, shape=(16, 12, 10))
    w.llg_max_iter, w.llg_tol = 2, 1e-30
    got, ref, gs, os_ = _run_both(w, 5)
    _assert_parity(got, ref, True)
    assert gs["nonconverged_halfsteps"] == 10 == int(os_["nonconverged"])
    assert gs["iters_total"] == 20
    w.llg_max_iter = 1            # odd and even caps exercise both Jacobi buffers
    got, ref, gs, _ = _run_both(w, 5)
    _assert_parity(got, ref, True)


def test_llg_enabled_without_magnetic_cells_is_plain_maxwell():
    w = wl.make_config(2, shape=(24, 10, 6), steps=20)
    w.enable_llg = True
    got, ref, gs, _ = _run_both(w, 20)
    _assert_parity(got, ref, True)
    assert gs["magnetic_cells"] == 0 and gs["iters_total"] == 0


def test_errors_are_reported_not_thrown_from_c():
    from paper_2103_12819_b200 import binding as B
    with pytest.raises(B.FdtdLlgError) as e:
        B.FdtdLlg(8, 8, 8, 1e-6, 1e-6, 1e-6, 1e-15, materials={"eps_r": torch.zeros(8, 8, 8, dtype=torch.float64)})
    assert e.value.code == B.EINVAL and "eps_r" in str(e.value)
    with pytest.raises(B.FdtdLlgError) as e:
        B.FdtdLlg(8, 8, 8, 1e-6, 1e-6, 1e-6, 1e-15, materials={"Ms": -torch.ones(8, 8, 8, dtype=torch.float64)})
    assert e.value.code == B.EINVAL and "Ms" in str(e.value)
    sim = B.FdtdLlg(8, 8, 8, 1e-6, 1e-6, 1e-6, 1e-15, materials={"Ms": 1e5, "gamma": 1.759e11})
    with pytest.raises(B.FdtdLlgError) as e:
        sim.set_fields()          # magnetic faces with no M direction
    assert e.value.code == B.EINVAL
    with pytest.raises(B.FdtdLlgError):
        sim.set_source(0, (0, 0, 0), (9, 8, 8))
    with pytest.raises(B.FdtdLlgError):
        sim.step(-1)
    st = sim.stats()
    assert st["courant"] == pytest.approx(1e-15 / wl.courant_dt(1.0, 1e-6, 1e-6, 1e-6))


def test_h_source_added_mid_run_leaves_the_merged_mode_and_restart_with_set_fields():
    """merge_h keeps H at half-integer time outside the sweep box; an H source acts on H at integer
    time, so adding one converts the state back (unmerge).  Oracle: the same source added after the
    same number of steps.  Then set_fields on the used handle gives what a fresh handle gives."""
    from paper_2103_12819_b200.binding import from_workload
    for cfg in (4, 3):
        w = wl.make_config(cfg, shape=wl.SMALL_SHAPES[cfg])
        o = oracle_from_workload(w)
        sim = from_workload(w)
        assert sim.stats()["merged_h"] == 1
        o.step(17)
        sim.step(17)
        f0, tp = 5e12, 20 * w.dt
        lo, hi = (3, 2, 5), (w.nx - 2, w.ny - 1, 9)
        o.set_source(1, lo, hi, None, 3e2, f0, 40 * w.dt, tp, kind=3)           # hard H_y
        sim.set_source(1, lo, hi, None, 3e2, f0, 40 * w.dt, tp, kind=3)
        assert sim.stats()["merged_h"] == 0
        o.step(25)
        sim.step(25)
        _assert_parity(_gpu_fields(sim), o.read_fields(), w.enable_llg)
        assert sim.stats()["steps"] == 42
    # restart: set_fields resets the clock, the statistics and the half-time state of the merged faces
    w = wl.make_config(4, shape=wl.SMALL_SHAPES[4])
    a, b = from_workload(w), from_workload(w)
    a.step(13)
    a.set_fields(w.E, w.H, w.M_cell)
    a.step(20)
    b.step(20)
    fa, fb = _gpu_fields(a), _gpu_fields(b)
    for k in fa:
        assert np.array_equal(fa[k], fb[k]), k
    assert a.stats()["steps"] == 20
