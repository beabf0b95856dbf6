"""Pins of the oracle's hard / soft field sources (reading A25 in DESIGN.md), CPU only.

S1  hard E source, closed form: in a vacuum column (ny = nz = 1, periodic) at the 1-D "magic" step
    c dt = dx the Yee scheme propagates E exactly one cell per step, so a hard source
    Ey(i0, n) = g(n dt) radiates Ey(i, n) = g((n - |i - i0|) dt) to rounding (discrete d'Alembert),
    and Hz = -/+ Ey / eta0 ... checked on E.  Pins the time argument (n+1) dt and "after the update".
S2  soft H source: the field is linear in the source; with the soft source alone (zero initial
    fields) doubling the amplitude doubles every field, and the first step's H equals
    dt A g(0) profile advanced by one step of the source-free scheme (superposition).
S3  all four kinds together against the 80-bit numpy restatement on 8^3, every BC mix, with walls
    cutting the source boxes (wall-tangential E and wall-normal H stay 0).
S4  soft current of eq. 11 (the source of the hot path, `source_at`), closed form: a periodic box
    with H = 0, E = 0, uniform eps and sigma and a current that is uniform in space keeps curl H = 0,
    so eq. 11 is the scalar recurrence
        E^{n+1} = (sigma/2 + eps/dt)^-1 [ -(sigma/2 - eps/dt) E^n - J((n+1/2) dt) ],
    J(t) = A exp(-(t-t0)^2 / (2 Tp^2)) cos(2 pi f0 t) (the envelope of eq. 31), written
    here from the paper.  Pins the time argument (n+1/2) dt, the minus sign and the envelope's
    2 Tp^2; a box-shaped profile on a PEC grid pins where the current lands (first step).
"""
import math

import numpy as np
import pytest

from oracle import Oracle
from tests._util import rel_linf
from tests.bruteforce_np import BruteForce
from tests.test_oracle_pins import _random_case

C0 = 299792458.0


def test_s1_hard_e_source_is_exact_dalembert_at_the_magic_step():
    nx, dx = 160, 1e-3
    dt = dx / C0
    A, tp = 3.0, 6 * dt
    t0 = 8 * tp
    o = Oracle(nx, 1, 1, dx, dx, dx, dt, bc=(1, 1, 1), enable_llg=False)
    i0 = 20
    o.set_source(1, (i0, 0, 0), (i0 + 1, 1, 1), None, A, 0.0, t0, tp, kind=1)
    N = 70                       # the two fronts have not met around the periodic box yet
    o.step(N)
    ey = o.read_fields(("Ey",))["Ey"][0, 0]
    g = lambda n: A * np.exp(-0.5 * ((n * dt - t0) / tp) ** 2)
    i = np.arange(nx)
    dist = np.minimum(np.abs(i - i0), nx - np.abs(i - i0))
    ref = g(N - dist)
    assert np.max(np.abs(ref)) > 0.5 * A                      # the pulse is on the grid
    assert np.max(np.abs(ey - ref)) < 1e-12 * A
    # the wrong time argument (n + 1/2) dt would miss by O(dt g')
    assert np.max(np.abs(ey - g(N - 0.5 - dist))) > 1e-3 * A


def test_s2_soft_h_source_superposition():
    shape, d = (6, 5, 4), (1e-3, 1.1e-3, 0.9e-3)
    dt = 0.9 / (C0 * math.sqrt(sum(1 / h ** 2 for h in d)))
    rng = np.random.default_rng(3)
    prof = rng.random(3 * 2 * 2)
    args = dict(comp=2, lo=(1, 2, 1), hi=(4, 4, 3), profile=prof, f0=1e9, t0=0.0, tp=50 * dt)

    def run(A, steps):
        o = Oracle(*shape, *d, dt, bc=(1, 0, 1), enable_llg=False)
        o.set_source(amplitude=A, kind=2, **args)
        o.step(steps)
        return o.read_fields()
    f1, f2 = run(1e9, 6), run(2e9, 6)
    for n in ("Ex", "Ey", "Ez", "Hx", "Hy", "Hz"):
        assert np.max(np.abs(f2[n] - 2 * f1[n])) <= 1e-13 * np.max(np.abs(f2["Hz"]))
    # step 0: H += dt A g(0) profile (g(0) = 1 here), then one source-free step
    o = Oracle(*shape, *d, dt, bc=(1, 0, 1), enable_llg=False)
    hz = np.zeros(shape[::-1])
    hz[1:3, 2:4, 1:4] = dt * 1e9 * prof.reshape(2, 2, 3)
    o.set_fields(H=[None, None, hz])
    o.step(1)
    ref = o.read_fields()
    got = run(1e9, 1)
    for g in ("E", "H"):
        assert rel_linf(got, ref, g) < 1e-14
    assert np.max(np.abs(got["Ex"])) > 0


@pytest.mark.parametrize("bc,magnetic", [((1, 1, 1), False), ((0, 0, 0), True), ((1, 0, 1), True)])
def test_s3_all_kinds_bruteforce_8cubed(bc, magnetic):
    shape = (8, 8, 8)
    d, dt, kw, E, H, Mc, opts, _ = _random_case(23, shape, bc, magnetic, False, True, False)
    rng = np.random.default_rng(5)
    srcs = []
    for kind, comp, lo, hi, A in ((0, 0, (0, 0, 0), (8, 3, 8), 1e12), (1, 1, (0, 0, 0), (3, 8, 4), 2e6),
                                  (2, 2, (2, 0, 0), (7, 8, 2), 4e17), (3, 0, (0, 1, 3), (2, 6, 8), 5e2),
                                  (1, 2, (5, 5, 0), (8, 8, 8), -1e6)):
        nb = int(np.prod([h - l for l, h in zip(lo, hi)]))
        srcs.append(dict(kind=kind, comp=comp, lo=lo, hi=hi, profile=rng.random(nb), amplitude=A,
                         f0=3e12, t0=2e-15, tp=3e-15))
    o = Oracle(*shape, *d, dt, llg_tol=1e-15, llg_max_iter=40, **kw, **opts)
    o.set_fields(E, H, Mc)
    bf = BruteForce(shape, d, dt, bc, kw.get("eps_r"), kw.get("sigma"), kw.get("mu_r"),
                    kw.get("Ms"), kw.get("alpha"), kw.get("gamma"), magnetic,
                    opts["h_bias"], opts["ani_hk"], opts["ani_axis"], iters=8)
    bf.set_fields(E, H, Mc)
    for s in srcs:
        o.set_source(**s)
        bf.add_source(**s)
    o.step(4)
    bf.step(4)
    got, ref = o.read_fields(), bf.fields()
    assert rel_linf(got, ref, "E") < 1e-11
    assert rel_linf(got, ref, "H") < 1e-11
    if magnetic:
        assert rel_linf(got, ref, "M") < 1e-13
    # each kind left its mark: dropping it changes the result
    for drop in range(1, 4):
        o2 = Oracle(*shape, *d, dt, llg_tol=1e-15, llg_max_iter=40, **kw, **opts)
        o2.set_fields(E, H, Mc)
        for s in srcs:
            if s["kind"] != drop:
                o2.set_source(**s)
        o2.step(4)
        assert rel_linf(o2.read_fields(), got, "E") > 1e-6, drop
    # wall-tangential E / wall-normal H inside a source box stay 0 on PEC axes
    if bc[2] == 0:
        assert np.all(got["Ey"][0, :, :] == 0)      # Ey on the k = 0 wall (box 1 covers it)
    if bc[0] == 0:
        assert np.all(got["Hx"][:, :, 0] == 0)      # Hx on the i = 0 wall (box 3 covers it)


EPS0 = 1.0 / (4.0e-7 * math.pi * C0 ** 2)


def _soft_current_recurrence(eps, sigma, dt, J, steps, shift=0.5, sign=-1.0):
    """Eq. 11 with curl H = 0, as printed: E^{n+1} = (s/2 + e/dt)^-1 [-(s/2 - e/dt) E^n - J^{n+1/2}]."""
    e, out = 0.0, []
    for n in range(steps):
        e = (-(sigma / 2 - eps / dt) * e + sign * J((n + shift) * dt)) / (sigma / 2 + eps / dt)
        out.append(e)
    return np.array(out)


@pytest.mark.parametrize("sigma", [0.0, 50.0])
def test_s4_soft_current_obeys_the_scalar_recurrence_of_eq_11(sigma):
    shape, d = (6, 5, 4), (1e-3, 1.2e-3, 0.8e-3)
    dt = 0.8 / (C0 * math.sqrt(sum(1 / h ** 2 for h in d)))
    eps_r, A, f0, tp = 2.5, 3.0e4, 1.0 / (17 * dt), 9 * dt
    t0 = 3 * tp                                    # eq. 31: the pulse is centred at 3 Tp
    n = shape[0] * shape[1] * shape[2]
    J = lambda t: A * math.exp(-(t - t0) ** 2 / (2 * tp ** 2)) * math.cos(2 * math.pi * f0 * t)
    steps = 50
    hist = {c: [] for c in range(3)}
    for comp in range(3):
        o = Oracle(*shape, *d, dt, eps_r=np.full(n, eps_r), sigma=np.full(n, sigma), bc=(1, 1, 1),
                   enable_llg=False)
        o.set_source(comp, (0, 0, 0), shape, None, A, f0, t0, tp, kind=0)
        for _ in range(steps):
            o.step(1)
            f = o.read_fields()
            e = f[("Ex", "Ey", "Ez")[comp]]
            assert np.all(e == e.flat[0])                          # uniform in space
            for other in ("Ex", "Ey", "Ez", "Hx", "Hy", "Hz"):      # nothing else moves
                if other != ("Ex", "Ey", "Ez")[comp]:
                    assert not np.any(f[other])
            hist[comp].append(float(e.flat[0]))
    ref = _soft_current_recurrence(eps_r * EPS0, sigma, dt, J, steps)
    scale = np.max(np.abs(ref))
    assert scale > 0.01 * A * dt / (eps_r * EPS0)                   # the pulse has acted
    for comp in range(3):
        assert np.max(np.abs(np.array(hist[comp]) - ref)) <= 1e-13 * scale, comp
    # what a slip would give: J at n dt or (n+1) dt, the opposite sign, the envelope with Tp^2
    got = np.array(hist[1])
    for wrong in (_soft_current_recurrence(eps_r * EPS0, sigma, dt, J, steps, shift=0.0),
                  _soft_current_recurrence(eps_r * EPS0, sigma, dt, J, steps, shift=1.0),
                  _soft_current_recurrence(eps_r * EPS0, sigma, dt, J, steps, sign=+1.0),
                  _soft_current_recurrence(eps_r * EPS0, sigma, dt,
                                           lambda t: A * math.exp(-(t - t0) ** 2 / tp ** 2)
                                           * math.cos(2 * math.pi * f0 * t), steps)):
        assert np.max(np.abs(got - wrong)) > 1e-3 * scale


def test_s4_soft_current_profile_lands_on_its_box_and_not_on_the_walls():
    """First step from zero fields on a PEC grid: E^1 = -(sigma/2 + eps/dt)^-1 A g(dt/2) profile on the
    comp-edges of the box, 0 elsewhere and on wall-tangential edges."""
    shape, d = (7, 6, 5), (1e-3, 1.2e-3, 0.8e-3)
    nx, ny, nz = shape
    dt = 0.8 / (C0 * math.sqrt(sum(1 / h ** 2 for h in d)))
    eps_r, sigma, A, f0, tp = 3.0, 20.0, 2.0e5, 1.0 / (11 * dt), 4 * dt
    t0 = 0.3 * dt
    n = nx * ny * nz
    rng = np.random.default_rng(8)
    g = A * math.exp(-(0.5 * dt - t0) ** 2 / (2 * tp ** 2)) * math.cos(2 * math.pi * f0 * 0.5 * dt)
    k = -1.0 / (sigma / 2 + eps_r * EPS0 / dt)
    for comp in range(3):
        lo, hi = (0, 1, 0), (5, ny, 4)                 # touches the lower x and z walls, the upper y end
        nb = [h - l for l, h in zip(lo, hi)]
        prof = 0.5 + rng.random((nb[2], nb[1], nb[0]))
        o = Oracle(*shape, *d, dt, eps_r=np.full(n, eps_r), sigma=np.full(n, sigma), bc=(0, 0, 0),
                   enable_llg=False)
        o.set_source(comp, lo, hi, prof.ravel(), A, f0, t0, tp, kind=0)
        o.step(1)
        f = o.read_fields()
        ref = np.zeros((nz, ny, nx))
        ref[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = k * g * prof
        # a comp-edge is tangential to the walls of the two other axes: index 0 there stays 0
        # (array axes are z, y, x: grid axis a is array axis 2 - a)
        for axis in range(3):
            if axis != comp:
                idx = [slice(None)] * 3
                idx[2 - axis] = 0
                ref[tuple(idx)] = 0.0
        e = f[("Ex", "Ey", "Ez")[comp]]
        assert np.max(np.abs(ref)) > 0
        assert np.max(np.abs(e - ref)) <= 1e-14 * np.max(np.abs(ref)), comp
        for other in range(3):
            if other != comp:
                assert not np.any(f[("Ex", "Ey", "Ez")[other]])
