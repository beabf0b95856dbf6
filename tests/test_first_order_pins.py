"""Pins of the oracle's FIRST-ORDER scheme (eqs. 6-14),
CPU only.  What fixes it, with no implementation to compare against:

F1  closed form: alpha = 0, uniform M, E = 0.  B = H + M is conserved (eqs. 9, 14), so M x H_eff =
    M x A with the fixed axis A = H_bias + H0 + M0.  One forward-Euler half-step adds a vector
    perpendicular to M and A of length c|A||M_perp|, c = mu0 |gamma| dt/2, and N(M) rescales:
    the azimuth advances by atan(c|A|) and tan(theta) grows by sqrt(1 + c^2|A|^2) per half-step --
    exactly.  (The trapezoidal scheme rotates by 2 atan(c|A|/2) and keeps theta: pin P5.)
F2  damping: first-order convergence to the continuous damped precession (error ratio 2 under
    step halving), theta decreasing (the sign of the alpha term).
F3  PAPER.md:300: in the paper's convergence test "the convergence rates for the M components
    dropped to first order".
F4  invariants: |M| = Ms, div(H + M) constant, eq. 9 on the normal component.
F5  brute force on 8^3 against the numpy restatement of eqs. 7, 9, 12, 14 as printed (80-bit).
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from tests._util import rel_linf
from tests.bruteforce_np import BruteForce
from tests.test_oracle_pins import (GAMMA, MU0, _coarsen, _paper_convergence_run, _random_case,
                                    _rotate, courant)
from paper_2103_12819_b200 import workloads as wl
from tests._util import oracle_from_workload


def _uniform(theta0, phi0, Ms, alpha, bias, dt_scale=1.0, h_is_minus_m=True, gamma=GAMMA):
    shape, d = (4, 3, 2), (1e-3, 1e-3, 1e-3)
    dt = courant(0.9, d) * dt_scale
    shp = shape[::-1]
    m0 = Ms * np.array([math.sin(theta0) * math.cos(phi0), math.sin(theta0) * math.sin(phi0),
                        math.cos(theta0)])
    o = Oracle(*shape, *d, dt, Ms=np.full(shp, Ms), alpha=np.full(shp, alpha),
               gamma=np.full(shp, gamma), bc=(1, 1, 1), enable_llg=True, h_bias=bias,
               time_scheme=1)
    H = [np.full(shp, -m0[c]) for c in range(3)] if h_is_minus_m else [None] * 3
    o.set_fields(H=H, M_cell=[np.full(shp, m0[c]) for c in range(3)])
    return o, m0, dt


@pytest.mark.parametrize("h_is_minus_m", [True, False])
@pytest.mark.parametrize("gamma_sign", [1.0, -1.0])
def test_f1_exact_euler_rotation(h_is_minus_m, gamma_sign):
    Ms, bias = 1.4e5, np.array([2e3, -1e3, 1e4])
    o, m0, dt = _uniform(0.4, 0.3, Ms, 0.0, tuple(bias), h_is_minus_m=h_is_minus_m,
                         gamma=gamma_sign * GAMMA)
    A = bias + (0 if h_is_minus_m else m0)
    nA = np.linalg.norm(A)
    N = 100
    o.step(N)
    c = MU0 * GAMMA * dt / 2
    ah = A / nA
    par, perp = (m0 @ ah) * ah, m0 - (m0 @ ah) * ah
    th0 = math.atan2(np.linalg.norm(perp), m0 @ ah)
    th = math.atan(math.tan(th0) * (1 + (c * nA) ** 2) ** N)          # 2N half-steps
    phi = 2 * N * math.atan(c * nA)
    e1 = perp / np.linalg.norm(perp)
    ref = Ms * (math.cos(th) * ah + math.sin(th) * _rotate(e1, A, phi))
    assert phi > 0.05 and th - th0 > 1e-6        # both effects are visible
    f = o.read_fields()
    for face in "xyz":
        got = np.array([f["M" + face + q].mean() for q in "xyz"])
        assert np.max(np.abs(got - ref)) / Ms < 5e-13
        wrong = Ms * (math.cos(th) * ah + math.sin(th) * _rotate(e1, A, -phi))
        assert np.max(np.abs(got - wrong)) / Ms > 1e-3                 # precession sense
        assert max(np.ptp(f["M" + face + q]) for q in "xyz") / Ms < 1e-14
    st = o.stats()
    assert st["iters_total"] == 2 * N and st["nonconverged"] == 0      # one sweep per half-step


def test_f2_damped_precession_first_order():
    Ms, hb, alpha, th0 = 1.4e5, 3e5, 0.2, 0.6
    errs = []
    for scale, N in ((1.0, 40), (0.5, 80), (0.25, 160)):
        o, m0, dt = _uniform(th0, 0.0, Ms, alpha, (0, 0, hb), dt_scale=scale)
        o.step(N)
        t = N * dt
        wp = MU0 * GAMMA * hb / (1 + alpha ** 2)
        th = 2 * math.atan(math.tan(th0 / 2) * math.exp(-alpha * wp * t))
        ph = wp * t
        ref = Ms * np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
        f = o.read_fields()
        got = np.array([f["Mz" + q].mean() for q in "xyz"])
        errs.append(np.max(np.abs(got - ref)) / Ms)
        assert abs(np.linalg.norm(got) / Ms - 1) < 1e-14
    assert 1e-6 < errs[0] < 5e-2
    assert 1.8 < errs[0] / errs[1] < 2.2 and 1.9 < errs[1] / errs[2] < 2.1
    assert th < th0 - 1e-3      # damping towards the field


@pytest.mark.slow
def test_f3_m_drops_to_first_order_in_the_papers_test():
    """PAPER.md:300.  Same set-up as Tab. 2 (pin P7) with the first-order coupling: the rates of
    the M components that carry the dynamics (My, Mz: M0 is along x) are ~1 (measured 1.02-1.07;
    the trapezoidal scheme gives 2.00 there), H is "more erratic" (1.6 for Hy, Hz), and the
    component along M0 stays at 2 (it only changes through |M| = Ms, at second order in the angle)."""
    import tests.test_oracle_pins as P
    orig = P.Oracle

    def first_order(*a, **k):
        return orig(*a, time_scheme=1, **k)
    P.Oracle = first_order
    try:
        sols = [_paper_convergence_run(n, s) for n, s in ((32, 5), (64, 10), (128, 20))]
    finally:
        P.Oracle = orig
    (c, _), (m, _), (f, _) = sols
    def rate(nm):
        e_cm = np.mean(np.abs(_coarsen(nm, m[nm]) - c[nm]))
        e_mf = np.mean(np.abs(_coarsen(nm, f[nm]) - m[nm]))
        return math.log2(e_cm / e_mf)
    for nm in ("Mxy", "Mxz", "Myy", "Myz", "Mzy", "Mzz"):
        assert 0.9 < rate(nm) < 1.2, (nm, rate(nm))
    for nm in ("Hy", "Hz"):
        assert 1.2 < rate(nm) < 1.9, (nm, rate(nm))


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 0)])
def test_f4_invariants(bc):
    w = wl.config1(shape=(12, 10, 8))
    w.bc = bc
    a = w.numpy()
    m = a["materials"]
    o = Oracle(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.dt, Ms=m["Ms"], alpha=m["alpha"],
               gamma=m["gamma"], bc=bc, enable_llg=True, h_bias=w.h_bias, time_scheme=1)
    o.set_fields(a["E"], a["H"], a["M_cell"])
    f0 = o.read_fields()
    o.step(25)
    f1 = o.read_fields()
    Ms = 1.4e5

    def div(f):
        out = 0
        for ax, c in zip((2, 1, 0), "xyz"):
            b = f["H" + c] + f["M" + c + c]
            if bc["xyz".index(c)]:
                nxt = np.roll(b, -1, axis=ax)
            else:                       # the upper wall face carries H + M = 0 (A13)
                nxt = np.concatenate([np.delete(b, 0, axis=ax), np.zeros_like(np.take(b, [0], axis=ax))], axis=ax)
            out = out + (nxt - b) / w.dx
        return out
    assert np.max(np.abs(div(f1) - div(f0))) < 1e-10 * Ms / w.dx
    for face in "xyz":
        nrm = np.sqrt(sum(f1["M" + face + q] ** 2 for q in "xyz"))
        mag = nrm > 0
        assert np.max(np.abs(nrm[mag] / Ms - 1)) < 1e-13
        assert mag.sum() > 0.5 * nrm.size
    assert max(np.max(np.abs(f1[n] - f0[n])) for n in ("Mxx", "Myy", "Mzz")) > 0


@pytest.mark.parametrize("bc,aniso,lossy,src", [((1, 1, 1), False, False, False),
                                                ((0, 0, 0), True, True, True),
                                                ((1, 0, 1), True, False, True)])
def test_f5_bruteforce_8cubed(bc, aniso, lossy, src):
    shape = (8, 8, 8)
    d, dt, kw, E, H, Mc, opts, sources = _random_case(17, shape, bc, True, aniso, lossy, src)
    o = Oracle(*shape, *d, dt, time_scheme=1, **kw, **opts)
    o.set_fields(E, H, Mc)
    bf = BruteForce(shape, d, dt, bc, kw.get("eps_r"), kw.get("sigma"), kw.get("mu_r"),
                    kw.get("Ms"), kw.get("alpha"), kw.get("gamma"), True,
                    opts["h_bias"], opts["ani_hk"], opts["ani_axis"], iters=1, scheme=1)
    bf.set_fields(E, H, Mc)
    for s in sources:
        o.set_source(**s)
        bf.add_source(**s)
    o.step(4)
    bf.step(4)
    got, ref = o.read_fields(), bf.fields()
    assert rel_linf(got, ref, "E") < 1e-11
    assert rel_linf(got, ref, "H") < 1e-11
    assert rel_linf(got, ref, "M") < 1e-13
    # and it is NOT the second-order scheme: the two differ at O(dt)
    o2 = Oracle(*shape, *d, dt, llg_tol=1e-15, llg_max_iter=40, **kw, **opts)
    o2.set_fields(E, H, Mc)
    for s in sources:
        o2.set_source(**s)
    o2.step(4)
    assert rel_linf(o2.read_fields(), ref, "M") > 1e-9


def test_literal_80bit_build_agrees_with_the_increment_form():
    """As A24 for the trapezoidal scheme: the increment-form fp64 evaluation of eqs. 7, 9 agrees
    with the 80-bit build to well under the 1e-9 parity bar."""
    w = wl.make_config(5, shape=(16, 16, 16))
    outs = []
    for kind in ("f64", "ld"):
        o = oracle_from_workload(w, kind)
        g = o._fn("set_scheme")
        g.argtypes = [type(o._h), __import__("ctypes").c_int]
        assert g(o._h, 1) == 0
        o.step(40)
        outs.append(o.read_fields())
    assert rel_linf(outs[0], outs[1], "E") < 5e-9
    assert rel_linf(outs[0], outs[1], "H") < 5e-9
    assert rel_linf(outs[0], outs[1], "M") < 1e-13
