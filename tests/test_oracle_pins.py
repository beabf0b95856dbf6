"""Pins of the CPU oracle to things other than itself (all CPU, ``-m "not gpu"``).

Each test states what it pins (P-numbers of DESIGN.md) and where the closed form comes from.
Constants and formulas are retyped here from the mathematics, not imported from ``oracle/``.
"""
import math
from pathlib import Path

import numpy as np
import pytest

from oracle import Oracle, constants
from tests._util import oracle_from_workload, rel_linf
from tests.bruteforce_np import BruteForce, shift
from paper_2103_12819_b200 import workloads as wl

MU0 = 4e-7 * math.pi
C0 = 299792458.0
EPS0 = 1.0 / (MU0 * C0 * C0)
ETA0 = math.sqrt(MU0 / EPS0)
GOLDEN = Path(__file__).resolve().parent / "golden"


def courant(cfl, d):
    return cfl / (C0 * math.sqrt(sum(1.0 / h ** 2 for h in d)))


def test_constants_consistent():
    c = constants()
    assert c["mu0"] == pytest.approx(MU0, rel=1e-15)
    assert 1.0 / math.sqrt(c["mu0"] * c["eps0"]) == pytest.approx(c["c0"], rel=1e-15)


# ----------------------------------------------------------------------------- P1 dispersion

def _positions(shape, d):
    nx, ny, nz = shape
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return [i * d[0], j * d[1], k * d[2]]


def _plane_wave(shape, d, dt, mvec, evec, t_steps):
    """Exact eigenmode of the scheme on a periodic vacuum grid (pin P1).

    E_a = e_a cos(k.r_a - w t) at the edge positions, with K_a = (2/d_a) sin(k_a d_a/2),
    e.K = 0, (2/dt) sin(w dt/2) = c |K| (the Yee numerical dispersion relation); leapfrog
    Faraday gives h = K x e / (mu0 W), W = (2/dt) sin(w dt/2); the scheme's integer-time H
    is the mean of H^{n+-1/2}, hence the factor cos(w dt/2)."""
    kvec = [2 * math.pi * m / (n * h) for m, n, h in zip(mvec, shape, d)]
    K = np.array([2 / h * math.sin(kk * h / 2) for kk, h in zip(kvec, d)])
    e = np.array(evec, float)
    e = e - K * (e @ K) / (K @ K)          # numerically divergence-free polarisation
    W = C0 * math.sqrt(K @ K)
    w = 2 / dt * math.asin(W * dt / 2)
    h = np.cross(K, e) / (MU0 * W) * math.cos(w * dt / 2)
    r = _positions(shape, d)
    t = t_steps * dt
    out = {}
    for a, nm in enumerate("xyz"):
        # edge a: +1/2 along a; face a: +1/2 along the two other axes
        ph_e = sum(kvec[b] * (r[b] + (0.5 * d[b] if b == a else 0.0)) for b in range(3))
        ph_h = sum(kvec[b] * (r[b] + (0.5 * d[b] if b != a else 0.0)) for b in range(3))
        out["E" + nm] = e[a] * np.cos(ph_e - w * t)
        out["H" + nm] = h[a] * np.cos(ph_h - w * t)
    return out, w


@pytest.mark.parametrize("mvec,evec", [((1, 0, 0), (0, 1, 0)), ((0, 2, 0), (0, 0, 1)),
                                       ((0, 0, 1), (1, 0, 0)), ((1, 2, 1), (1, -1, 0.5)),
                                       ((2, -1, 3), (0.3, 1, 1))])
def test_p1_yee_eigenmode_exact(mvec, evec):
    shape, d = (12, 10, 8), (1e-6, 1.3e-6, 0.7e-6)
    dt = courant(0.9, d)
    f0, w = _plane_wave(shape, d, dt, mvec, evec, 0)
    o = Oracle(*shape, *d, dt, bc=(1, 1, 1), enable_llg=False)
    o.set_fields([f0["Ex"], f0["Ey"], f0["Ez"]], [f0["Hx"], f0["Hy"], f0["Hz"]])
    N = 150
    o.step(N)
    got = o.read_fields()
    ref, _ = _plane_wave(shape, d, dt, mvec, evec, N)
    for nm in ("Ex", "Ey", "Ez"):
        assert np.max(np.abs(got[nm] - ref[nm])) < 2e-12
    for nm in ("Hx", "Hy", "Hz"):
        assert np.max(np.abs(got[nm] - ref[nm])) < 2e-12 / ETA0 * 3


def test_p1_config2_dispersion_numbers():
    """Config 2's mode: lambda = 32 cells at 0.9 Courant -> c dt/dx = 0.9/sqrt(3),
    w dt = 2 asin(0.9/sqrt3 sin(pi/32)); the noise-free twin equals cos(k i dx - N w dt)."""
    w = wl.make_config(2, shape=(32, 4, 4), steps=100, noise=0.0)
    wdt = 2 * math.asin(0.9 / math.sqrt(3) * math.sin(math.pi / 32))
    assert wdt == pytest.approx(0.10190649, abs=5e-9)   # value quoted in SURVEY.md 8(c).5-P1
    o = oracle_from_workload(w)
    o.step(100)
    got = o.read_fields(("Ey", "Hz"))
    i = np.arange(32)
    assert np.max(np.abs(got["Ey"][0, 0] - np.cos(2 * math.pi * i / 32 - 100 * wdt))) < 1e-12
    hz = math.cos(wdt / 2) / ETA0 * np.cos(2 * math.pi * (i + 0.5) / 32 - 100 * wdt)
    assert np.max(np.abs(got["Hz"][0, 0] - hz)) < 1e-14


# ----------------------------------------------------------------------------- P2 energy

def _np_curl_faces(E, d, per):
    out = []
    for a in range(3):
        a1, a2 = (a + 1) % 3, (a + 2) % 3
        out.append((shift(E[a2], a1, 1, per[a1]) - E[a2]) / d[a1]
                   - (shift(E[a1], a2, 1, per[a2]) - E[a1]) / d[a2])
    return out


def _edge_mean(a, dd, per):
    t1, t2 = (dd + 1) % 3, (dd + 2) % 3
    s1 = shift(a, t1, -1, per[t1])
    return (a + s1 + shift(a, t2, -1, per[t2]) + shift(s1, t2, -1, per[t2])) / 4


@pytest.mark.parametrize("bc", [(1, 1, 1), (0, 0, 0), (1, 0, 1), (0, 1, 0)])
def test_p2_leapfrog_energy_invariant(bc):
    """W = sum eps|E|^2 + mu0 sum|H|^2 - dt^2/(4 mu0) sum|curl E|^2 is conserved to round-off
    for any lossless dielectric and any mix of PEC/periodic axes (the naive energy is not)."""
    rng = np.random.default_rng(7)
    shape, d = (9, 7, 6), (1e-6, 0.8e-6, 1.2e-6)
    shp = shape[::-1]
    dt = courant(0.9, d)
    eps_r = 1 + 3 * rng.random(shp)
    E0 = [rng.standard_normal(shp) for _ in range(3)]
    H0 = [rng.standard_normal(shp) / ETA0 for _ in range(3)]
    o = Oracle(*shape, *d, dt, eps_r=eps_r, bc=bc, enable_llg=False)
    o.set_fields(E0, H0)

    def W(f):
        E = [f["Ex"], f["Ey"], f["Ez"]]
        H = [f["Hx"], f["Hy"], f["Hz"]]
        cu = _np_curl_faces(E, d, bc)
        return (sum(np.sum(EPS0 * _edge_mean(eps_r, a, bc) * E[a] ** 2) for a in range(3))
                + MU0 * sum(np.sum(h ** 2) for h in H)
                - dt * dt / (4 * MU0) * sum(np.sum(c ** 2) for c in cu))

    def naive(f):
        return (sum(np.sum(EPS0 * _edge_mean(eps_r, a, bc) * f["E" + c] ** 2)
                    for a, c in enumerate("xyz")) + MU0 * sum(np.sum(f["H" + c] ** 2) for c in "xyz"))

    f0 = o.read_fields()
    w0, n0 = W(f0), naive(f0)
    drift, ndrift = 0.0, 0.0
    for _ in range(10):
        o.step(20)
        f = o.read_fields()
        drift = max(drift, abs(W(f) - w0) / w0)
        ndrift = max(ndrift, abs(naive(f) - n0) / n0)
    assert drift < 5e-14
    assert ndrift > 1e-3   # shows the test has teeth: the naive energy does move


# ----------------------------------------------------------------------------- P3 PEC

@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p3_pec_cavity_mode(axis):
    """E_a = sin(m pi p/n_b) sin(n pi q/n_c) (a = axis, b,c the others), H = 0 is an exact
    eigenmode of the PEC box: E^N = cos(N w dt) E^0 with the Yee dispersion relation."""
    shape, d = (12, 16, 10), (1e-6, 1.1e-6, 0.9e-6)
    dt = courant(0.9, d)
    b, c = (axis + 1) % 3, (axis + 2) % 3
    mb, mc = 2, 3
    r = _positions(shape, (1, 1, 1))
    E0 = np.sin(mb * math.pi * r[b] / shape[b]) * np.sin(mc * math.pi * r[c] / shape[c])
    kb, kc = mb * math.pi / (shape[b] * d[b]), mc * math.pi / (shape[c] * d[c])
    s = C0 * dt * math.sqrt((math.sin(kb * d[b] / 2) / d[b]) ** 2 + (math.sin(kc * d[c] / 2) / d[c]) ** 2)
    wdt = 2 * math.asin(s)
    E = [None, None, None]
    E[axis] = E0
    o = Oracle(*shape, *d, dt, bc=(0, 0, 0), enable_llg=False)
    o.set_fields(E)
    N = 300
    o.step(N)
    f = o.read_fields()
    names = ["Ex", "Ey", "Ez"]
    assert np.max(np.abs(f[names[axis]] - math.cos(N * wdt) * E0)) < 1e-12
    assert np.max(np.abs(f[names[b]])) == 0.0 and np.max(np.abs(f[names[c]])) == 0.0


def test_pec_reflection_coefficient_minus_one():
    """a wave reflected by an infinite PEC wall has reflection coefficient -1.
    Method of images: the PEC run on n cells equals the odd-image run on a periodic 2n grid."""
    n, d = 64, (1e-6, 1e-6, 1e-6)
    dt = courant(0.9, d)
    i = np.arange(2 * n)
    pulse = lambda x: np.exp(-((x - 40.0) / 5.0) ** 2)
    ey = pulse(i) - pulse(2 * n - i)                 # odd about 0 and n
    hz = (pulse(i + 0.5) + pulse(2 * n - i - 0.5)) / ETA0   # even image of a +x going wave
    big = Oracle(2 * n, 1, 1, *d, dt, bc=(1, 1, 1), enable_llg=False)
    big.set_fields([None, ey.reshape(1, 1, -1), None], [None, None, hz.reshape(1, 1, -1)])
    box = Oracle(n, 1, 1, *d, dt, bc=(0, 1, 1), enable_llg=False)
    box.set_fields([None, ey[:n].reshape(1, 1, -1), None], [None, None, hz[:n].reshape(1, 1, -1)])
    big.step(120)
    box.step(120)   # the pulse has hit the wall at x = n and travels back inverted
    fb, fx = big.read_fields(("Ey", "Hz")), box.read_fields(("Ey", "Hz"))
    assert np.max(np.abs(fx["Ey"][0, 0] - fb["Ey"][0, 0, :n])) < 1e-14
    assert np.max(np.abs(fx["Hz"][0, 0] - fb["Hz"][0, 0, :n])) < 1e-14 / ETA0 * 10
    # and the reflected pulse really is there, inverted
    assert fx["Ey"][0, 0].min() < -0.4 and fx["Ey"][0, 0].max() < 0.2


# ----------------------------------------------------------------------------- P4 sigma

@pytest.mark.parametrize("sigma,eps_r", [(50.0, 2.0), (5.8e7, 1.0)])
def test_p4_uniform_conductor_decay(sigma, eps_r):
    """Uniform E, H = 0, periodic: E^N = Ca^N E^0, Ca = (2 eps - sigma dt)/(2 eps + sigma dt)."""
    shape, d = (4, 3, 5), (1e-6, 1e-6, 1e-6)
    dt = courant(0.9, d)
    shp = shape[::-1]
    o = Oracle(*shape, *d, dt, eps_r=np.full(shp, eps_r), sigma=np.full(shp, sigma),
               bc=(1, 1, 1), enable_llg=False)
    o.set_fields([np.full(shp, v) for v in (1.0, -2.0, 3.0)])
    N = 25
    o.step(N)
    eps = EPS0 * eps_r
    Ca = (2 * eps - sigma * dt) / (2 * eps + sigma * dt)
    f = o.read_fields(("Ex", "Ey", "Ez"))
    for nm, v in zip(("Ex", "Ey", "Ez"), (1.0, -2.0, 3.0)):
        assert np.allclose(f[nm], v * Ca ** N, rtol=1e-12, atol=0)
    if sigma > 1e6:
        assert Ca == pytest.approx(-0.999648, abs=2e-6)   # copper at 1 um, SURVEY.md P4


def test_p4_lossy_mode_three_term_recurrence():
    """A divergence-free Fourier mode in a uniform lossy medium obeys
    E^{n+2} - B E^{n+1} + Ca E^n = 0, B = 1 + Ca - Cb dt K^2/mu0, Cb = 2dt/(2eps+sigma dt)."""
    shape, d = (8, 6, 10), (1e-6, 1.2e-6, 0.9e-6)
    dt = courant(0.9, d)
    shp = shape[::-1]
    sigma, eps_r = 50.0, 2.0
    mvec = (1, -1, 2)
    f0, _ = _plane_wave(shape, d, dt, mvec, (1, 0.5, -0.2), 0)
    o = Oracle(*shape, *d, dt, eps_r=np.full(shp, eps_r), sigma=np.full(shp, sigma),
               bc=(1, 1, 1), enable_llg=False)
    o.set_fields([f0["Ex"], f0["Ey"], f0["Ez"]], [f0["Hx"], f0["Hy"], f0["Hz"]])
    hist = []
    for _ in range(6):
        hist.append(o.read_fields(("Ex", "Ey", "Ez")))
        o.step(1)
    eps = EPS0 * eps_r
    Ca = (2 * eps - sigma * dt) / (2 * eps + sigma * dt)
    Cb = 2 * dt / (2 * eps + sigma * dt)
    K2 = sum((2 / h * math.sin(math.pi * m / n)) ** 2 for m, n, h in zip(mvec, shape, d))
    B = 1 + Ca - Cb * dt * K2 / MU0
    for n in range(4):
        for nm in ("Ex", "Ey", "Ez"):
            res = hist[n + 2][nm] - B * hist[n + 1][nm] + Ca * hist[n][nm]
            assert np.max(np.abs(res)) < 1e-13


def test_dielectric_slows_the_wave():
    """P1 in a uniform dielectric: c -> c/sqrt(eps_r)."""
    shape, d = (16, 2, 2), (1e-6, 1e-6, 1e-6)
    dt = courant(0.9, d)
    eps_r = 11.7
    k = 2 * math.pi / (16 * d[0])
    wdt = 2 * math.asin(C0 / math.sqrt(eps_r) * dt / d[0] * math.sin(k * d[0] / 2))
    i = np.arange(16)
    ey = np.cos(k * d[0] * i)
    hz = math.cos(wdt / 2) * math.sqrt(eps_r) / ETA0 * np.cos(k * d[0] * (i + 0.5))
    shp = shape[::-1]
    o = Oracle(*shape, *d, dt, eps_r=np.full(shp, eps_r), bc=(1, 1, 1), enable_llg=False)
    o.set_fields([None, np.broadcast_to(ey, shp), None], [None, None, np.broadcast_to(hz, shp)])
    o.step(200)
    f = o.read_fields(("Ey",))
    assert np.max(np.abs(f["Ey"][0, 0] - np.cos(k * d[0] * i - 200 * wdt))) < 1e-12


# ----------------------------------------------------------------------------- P5/P6/P9 LLG

GAMMA = 1.759e11


def _uniform_magnet(theta0, phi0, Ms, alpha, bias, dt_scale=1.0, hk=0.0, h_is_minus_m=True,
                    tol=1e-14, dx=1e-3, gamma=GAMMA):
    shape, d = (4, 3, 2), (dx, dx, dx)
    dt = courant(0.9, d) * dt_scale
    shp = shape[::-1]
    m0 = Ms * np.array([math.sin(theta0) * math.cos(phi0), math.sin(theta0) * math.sin(phi0),
                        math.cos(theta0)])
    o = Oracle(*shape, *d, dt, Ms=np.full(shp, Ms), alpha=np.full(shp, alpha),
               gamma=np.full(shp, gamma), bc=(1, 1, 1), enable_llg=True, h_bias=bias,
               ani_hk=hk, llg_tol=tol, llg_max_iter=60)
    H = [np.full(shp, -m0[c]) for c in range(3)] if h_is_minus_m else [None] * 3
    o.set_fields(H=H, M_cell=[np.full(shp, m0[c]) for c in range(3)])
    return o, m0, dt


def _rotate(v, axis, ang):
    axis = axis / np.linalg.norm(axis)
    return (v * math.cos(ang) + np.cross(axis, v) * math.sin(ang)
            + axis * (axis @ v) * (1 - math.cos(ang)))


@pytest.mark.parametrize("h_is_minus_m", [True, False])
@pytest.mark.parametrize("gamma_sign", [1.0, -1.0])
def test_p5_exact_cayley_larmor_rotation(h_is_minus_m, gamma_sign):
    """alpha = 0, uniform M, E = 0: B is conserved, H = H0 + M0 - M, so M precesses about
    A = H_bias + H0 + M0 and each converged trapezoidal half-step is an exact rotation by
    2 atan(mu0 |gamma| |A| dt/4), counter-clockwise about A (dM/dt = -mu0|gamma| M x H).
    With H0 = -M0 this is textbook Larmor precession about the bias (north_star's check)."""
    Ms, bias = 1.4e5, np.array([2e3, -1e3, 1e4])
    o, m0, dt = _uniform_magnet(0.4, 0.3, Ms, 0.0, tuple(bias), h_is_minus_m=h_is_minus_m,
                                gamma=gamma_sign * GAMMA)
    A = bias + (0 if h_is_minus_m else m0)
    N = 100
    o.step(N)
    ang = 2 * N * 2 * math.atan(MU0 * GAMMA * np.linalg.norm(A) * dt / 4)
    ref = _rotate(m0, A, ang)
    assert ang > 0.05                           # a visible rotation, not a null test
    f = o.read_fields()
    for face in "xyz":
        got = np.array([f["M" + face + c].mean() for c in "xyz"])
        assert np.max(np.abs(got - ref)) / Ms < 5e-13
        # the wrong precession sense would miss by O(ang)
        assert np.max(np.abs(got - _rotate(m0, A, -ang))) / Ms > 1e-3
        spread = max(np.ptp(f["M" + face + c]) for c in "xyz")
        assert spread / Ms < 1e-14
    # H followed M: H = H0 + M0 - M on every face (eq. 21 with curl E = 0)
    h0 = -m0 if h_is_minus_m else np.zeros(3)
    for a, face in enumerate("xyz"):
        assert abs(f["H" + face].mean() - (h0[a] + m0[a] - ref[a])) / Ms < 5e-13
    assert o.stats()["nonconverged"] == 0


def test_p9_anisotropy_axis_field():
    """u = z, H_bias || z, alpha = 0: m_z is constant, the axis field is H_bias + H_k m_z and the
    rotation per half-step is 2 atan(mu0|gamma|(H_bias + H_k m_z) dt/4) about z (reading A19)."""
    Ms, hb, hk, th0 = 1.4e5, 8e4, 2e3, math.radians(5.0)
    o, m0, dt = _uniform_magnet(th0, 0.0, Ms, 0.0, (0, 0, hb), hk=hk)
    N = 100
    o.step(N)
    ang = 2 * N * 2 * math.atan(MU0 * GAMMA * (hb + hk * math.cos(th0)) * dt / 4)
    ref = _rotate(m0, np.array([0, 0, 1.0]), ang)
    noani = _rotate(m0, np.array([0, 0, 1.0]),
                    2 * N * 2 * math.atan(MU0 * GAMMA * hb * dt / 4))
    f = o.read_fields()
    got = np.array([f["Mx" + c].mean() for c in "xyz"])
    assert np.max(np.abs(got - ref)) / Ms < 5e-13
    assert np.max(np.abs(got - noani)) / Ms > 1e-4     # the H_k term is visible


def test_p6_damped_precession_second_order():
    """alpha > 0, H0 = -M0: tan(theta/2) = tan(theta0/2) exp(-alpha w' t), phi = w' t,
    w' = mu0|gamma|H/(1+alpha^2).  The scheme is second order: error ratio 4 under dt halving."""
    Ms, hb, alpha, th0 = 1.4e5, 3e5, 0.2, 0.6
    errs = []
    for scale, N in ((1.0, 40), (0.5, 80), (0.25, 160)):
        o, m0, dt = _uniform_magnet(th0, 0.0, Ms, alpha, (0, 0, hb), dt_scale=scale)
        o.step(N)
        t = N * dt
        wp = MU0 * GAMMA * hb / (1 + alpha ** 2)
        th = 2 * math.atan(math.tan(th0 / 2) * math.exp(-alpha * wp * t))
        ph = wp * t
        ref = Ms * np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
        f = o.read_fields()
        got = np.array([f["Mz" + c].mean() for c in "xyz"])
        errs.append(np.max(np.abs(got - ref)) / Ms)
        assert abs(np.linalg.norm(got) / Ms - 1) < 1e-14
    assert errs[0] < 1e-3 and errs[0] > 1e-9
    assert 3.8 < errs[0] / errs[1] < 4.2 and 3.8 < errs[1] / errs[2] < 4.2
    # damping really happened (theta decreased measurably)
    assert th < th0 - 1e-3


# ----------------------------------------------------------------------------- P8 invariants

def _cfg1_like(shape=(12, 10, 8), bc=(0, 0, 0), steps=0, seed_shift=0):
    w = wl.config1(shape=shape)
    w.bc = bc
    return w


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 0), (1, 1, 1)])
def test_p8_norm_and_divergence_invariants(bc):
    """(i) |M| = Ms_f on every magnetic face; (ii) discrete div(H + M) is constant
    in time in every cell where mu = mu0 (eq. 21 changes H + M by a discrete curl only)."""
    w = _cfg1_like(bc=bc)
    o = oracle_from_workload(w)
    d = (w.dx, w.dy, w.dz)

    def div_b(f):
        tot = 0
        for a, c in enumerate("xyz"):
            b = f["H" + c] + f["M" + c + c]
            tot = tot + (shift(b, a, 1, bc[a]) - b) / d[a]
        return tot

    f0 = o.read_fields()
    div0 = div_b(f0)
    o.step(30)
    f = o.read_fields()
    Ms = 1.4e5
    for face, a in zip("xyz", range(3)):
        nrm = np.sqrt(sum(f["M" + face + c] ** 2 for c in "xyz"))
        idx = np.indices(nrm.shape)[2 - a]
        wall = (idx == 0) if not bc[a] else np.zeros_like(nrm, bool)
        assert np.max(np.abs(nrm[~wall] / Ms - 1)) < 1e-13
        assert np.all(nrm[wall] == 0)              # A13: wall faces carry no M
    assert np.max(np.abs(div_b(f) - div0)) * d[0] / Ms < 1e-13
    # M moved (the invariants are not trivially true)
    assert max(np.max(np.abs(f["Mx" + c] - f0["Mx" + c])) for c in "xyz") / Ms > 1e-9
    st = o.stats()
    assert st["nonconverged"] == 0 and 2 <= st["iters_max"] <= 5


def test_p8_accepted_iterate_satisfies_eq15():
    """The accepted M^{n+1/2} satisfies the trapezoidal LLG equation (15) up to the
    renormalisation and tol.  Residual written from eq. 15 itself, not from eq. 18."""
    shape, bc = (6, 5, 4), (1, 1, 1)
    dx = 1e-3                                    # large cell => large dt => visible LLG dynamics
    rng = np.random.default_rng(3)
    shp = shape[::-1]
    Ms, alpha = 1.4e5, 0.05
    dt = courant(0.9, (dx, dx, dx))
    o = Oracle(*shape, dx, dx, dx, dt, Ms=np.full(shp, Ms), alpha=np.full(shp, alpha),
               gamma=np.full(shp, -GAMMA), bc=bc, h_bias=(0, 0, 1e4), llg_tol=1e-15,
               llg_max_iter=80)
    th = 0.5 * rng.random(shp)
    ph = 2 * math.pi * rng.random(shp)
    Mc = [Ms * np.sin(th) * np.cos(ph), Ms * np.sin(th) * np.sin(ph), Ms * np.cos(th)]
    H0 = [1e3 * rng.standard_normal(shp) for _ in range(3)]
    E0 = [1e5 * rng.standard_normal(shp) for _ in range(3)]
    o.set_fields(E0, H0, Mc)
    f0 = o.read_fields()
    o.hm_half_step()
    f1 = o.read_fields()
    assert o.stats()["nonconverged"] == 0

    def heff(f, face, a):
        out = []
        for t, c in enumerate("xyz"):
            if t == a:
                h = f["H" + c]
            else:
                a0 = f["H" + c]
                a1 = shift(a0, a, -1, True)
                h = 0.25 * (a0 + a1 + shift(a0, t, 1, True) + shift(a1, t, 1, True))
            out.append(h + (1e4 if t == 2 else 0.0))
        return out

    cr = lambda u, v: [u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0]]
    g = -GAMMA   # the electron's negative gamma, as in eq. 3
    for a, face in enumerate("xyz"):
        m0 = [f0["M" + face + c] for c in "xyz"]
        m1 = [f1["M" + face + c] for c in "xyz"]
        h0, h1 = heff(f0, face, a), heff(f1, face, a)
        t0, t1 = cr(m0, h0), cr(m1, h1)
        mid = [(u + v) / 2 for u, v in zip(m0, m1)]
        rate = [(v - u) / (dt / 2) for u, v in zip(m0, m1)]
        damp = cr(mid, rate)
        for q in range(3):
            res = rate[q] - (MU0 * g / 2) * (t0[q] + t1[q]) - alpha / Ms * damp[q]
            scale = np.max(np.abs(rate[q])) + 1e-300
            # renormalisation perturbs M^{n+1/2} at O(|dM|^2/Ms) only
            assert np.max(np.abs(res)) / scale < 5e-4
    # and the H update is eq. 21: H1 - H0 + M1 - M0 = -(dt/2mu0) curl E  on the normal component
    cu = _np_curl_faces(E0, (dx, dx, dx), bc)
    for a, c in enumerate("xyz"):
        lhs = f1["H" + c] - f0["H" + c] + f1["M" + c + c] - f0["M" + c + c]
        assert np.max(np.abs(lhs + dt / (2 * MU0) * cu[a])) < 1e-9 * np.max(np.abs(dt / (2 * MU0) * cu[a]))


# ----------------------------------------------------------------------------- P7 convergence

def _paper_convergence_run(n, steps, kind="f64"):
    """periodic L = 0.1 box centred at 0, eqs. 22-28, M = (Ms,0,0), CFL 0.9."""
    L = 0.1
    h = L / n
    dt = courant(0.9, (h, h, h))
    c = -L / 2 + (np.arange(n) + 0.5) * h      # cell centres
    e = -L / 2 + np.arange(n) * h              # nodes
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    g = np.exp(-1000 * (X ** 2 + Y ** 2 + Z ** 2))
    Ms = 1e4 * (1 + g)
    b = lambda arr, ax: np.broadcast_to(arr.reshape([n if q == ax else 1 for q in range(3)]), (n, n, n))
    # numpy axes: 0 = z, 1 = y, 2 = x
    Ex = 1e6 * np.cos(20 * math.pi * b(e, 0))            # Ex(z) at (i+1/2, j, k): z = node
    Ey = 1e6 * np.cos(20 * math.pi * b(e, 2))            # Ey(x) at (i, j+1/2, k)
    Ez = 1e6 * np.cos(20 * math.pi * b(e, 1))            # Ez(y) at (i, j, k+1/2)
    Hx = 1e6 / (120 * math.pi) * np.cos(20 * math.pi * b(c, 1))   # Hx(y) at (i, j+1/2, k+1/2)
    Hy = 1e6 / (120 * math.pi) * np.cos(20 * math.pi * b(c, 0))   # Hy(z) at (i+1/2, j, k+1/2)
    Hz = 1e6 / (120 * math.pi) * np.cos(20 * math.pi * b(c, 2))   # Hz(x) at (i+1/2, j+1/2, k)
    o = Oracle(n, n, n, h, h, h, dt, eps_r=1 + g, sigma=0.1 * g, Ms=Ms, alpha=0.5 * (1 + g),
               gamma=-1.759e11 * (1 + g), bc=(1, 1, 1), enable_llg=True, llg_tol=1e-6,
               llg_max_iter=50, kind=kind)
    o.set_fields([Ex, Ey, Ez], [Hx, Hy, Hz], [Ms, None, None])
    o.step(steps)
    return o.read_fields(), o.stats()


def _coarsen(name, a):
    """Average the fine values overlying each coarse edge / face."""
    kind, comp = name[0], "xyz".index(name[1])
    ax = {0: 2, 1: 1, 2: 0}
    out = a
    for d in range(3):
        along = (d == comp)
        # edge comp: two fine edges along its own axis, none across; face comp: four fine faces
        avg = along if kind == "E" else (not along)
        n = out.shape[ax[d]]
        sl0 = [slice(None)] * 3
        sl1 = [slice(None)] * 3
        sl0[ax[d]] = slice(0, n, 2)
        sl1[ax[d]] = slice(1, n, 2)
        out = 0.5 * (out[tuple(sl0)] + out[tuple(sl1)]) if avg else out[tuple(sl0)]
    return out


@pytest.mark.slow
def test_p7_second_order_convergence_paper_table2():
    """PAPER.md:286-298 (Tab. 2): rates 1.99-2.00 for all of E, H, M on 32/64/128 grids run 5/10/20
    steps.  Golden rates come from the paper (tests/golden/table2_rates.txt); the absolute L1
    values of Tab. 2 are unpinned, so only the rates are compared."""
    golden = {}
    for line in (GOLDEN / "table2_rates.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            golden[k] = float(v)
    sols = [_paper_convergence_run(n, s) for n, s in ((32, 5), (64, 10), (128, 20))]
    for _, st in sols:
        assert st["nonconverged"] == 0
    names = {"Ex": "Ex", "Ey": "Ey", "Ez": "Ez", "Hx": "Hx", "Hy": "Hy", "Hz": "Hz",
             "Mx": "Mxx", "My": "Myy", "Mz": "Mzz"}
    (c, _), (m, _), (f, _) = sols
    for label, nm in names.items():
        e_cm = np.mean(np.abs(_coarsen(nm, m[nm]) - c[nm]))
        e_mf = np.mean(np.abs(_coarsen(nm, f[nm]) - m[nm]))
        rate = math.log2(e_cm / e_mf)
        assert abs(rate - golden[label]) < 0.08, (label, rate)
    # every one of the 9 M components converges at second order too
    for nm in ("Mxy", "Mxz", "Myx", "Myz", "Mzx", "Mzy"):
        e_cm = np.mean(np.abs(_coarsen(nm, m[nm]) - c[nm]))
        e_mf = np.mean(np.abs(_coarsen(nm, f[nm]) - m[nm]))
        assert abs(math.log2(e_cm / e_mf) - 2.0) < 0.1, nm


# ----------------------------------------------------------------------------- P10 brute force

def _random_case(seed, shape, bc, magnetic, aniso, lossy, src):
    rng = np.random.default_rng(seed)
    shp = shape[::-1]
    d = (1e-6, 1.2e-6, 0.8e-6)
    dt = courant(0.9, d)
    kw = {}
    if lossy:
        kw["eps_r"] = 1 + 3 * rng.random(shp)
        kw["sigma"] = 100 * rng.random(shp) * (rng.random(shp) < 0.5)
        kw["mu_r"] = 1 + rng.random(shp) * (rng.random(shp) < 0.3)
    Mc = [None] * 3
    if magnetic:
        Ms = 1.4e5 * (1 + rng.random(shp)) * (rng.random(shp) < 0.6)
        kw["Ms"] = Ms
        kw["alpha"] = 0.01 + 0.05 * rng.random(shp)
        kw["gamma"] = -GAMMA * (1 + 0.1 * rng.random(shp))
        if "mu_r" in kw:
            kw["mu_r"] = np.where(Ms > 0, 1.0, kw["mu_r"])
        th, ph = math.pi * rng.random(shp), 2 * math.pi * rng.random(shp)
        Mc = [Ms * np.sin(th) * np.cos(ph), Ms * np.sin(th) * np.sin(ph), Ms * np.cos(th)]
    E = [1e6 * rng.standard_normal(shp) for _ in range(3)]
    H = [1e3 * rng.standard_normal(shp) for _ in range(3)]
    opts = dict(bc=bc, enable_llg=magnetic, h_bias=(1e3, -2e3, 1e4),
                ani_hk=(3e3 if aniso else 0.0), ani_axis=(0.6, 0.0, 0.8))
    sources = []
    if src:
        lo, hi = (1, 2, 1), (shape[0] - 1, 5, 4)
        nb = int(np.prod([h - l for l, h in zip(lo, hi)]))
        sources.append(dict(comp=1, lo=lo, hi=hi, profile=rng.random(nb), amplitude=1e12,
                            f0=2e12, t0=3e-15, tp=2e-15))
        sources.append(dict(comp=2, lo=(0, 0, 0), hi=shape, profile=None, amplitude=5e11,
                            f0=1e12, t0=1e-15, tp=4e-15))
    return d, dt, kw, E, H, Mc, opts, sources


@pytest.mark.parametrize("bc,magnetic,aniso,lossy,src", [
    ((1, 1, 1), False, False, False, False),
    ((0, 0, 0), False, False, True, True),
    ((1, 0, 1), True, False, False, False),
    ((0, 0, 0), True, True, True, True),
    ((1, 1, 0), True, True, False, True),
    ((0, 1, 1), True, False, True, False),
])
def test_p10_bruteforce_8cubed(bc, magnetic, aniso, lossy, src):
    """Oracle (C, per-point, increment form, fp64) vs an 80-bit whole-array numpy evaluation of
    the printed formulas, 4 steps on random 8^3 inputs."""
    shape = (8, 8, 8)
    d, dt, kw, E, H, Mc, opts, sources = _random_case(11, shape, bc, magnetic, aniso, lossy, src)
    o = Oracle(*shape, *d, dt, llg_tol=1e-15, llg_max_iter=40, **kw, **opts)
    o.set_fields(E, H, Mc)
    bf = BruteForce(shape, d, dt, bc, kw.get("eps_r"), kw.get("sigma"), kw.get("mu_r"),
                    kw.get("Ms"), kw.get("alpha"), kw.get("gamma"), magnetic,
                    opts["h_bias"], opts["ani_hk"], opts["ani_axis"], iters=8)
    bf.set_fields(E, H, Mc)
    for s in sources:
        o.set_source(**s)
        bf.add_source(**s)
    f0, b0 = o.read_fields(), bf.fields()
    for grp in ("E", "H", "M"):
        assert rel_linf(f0, b0, grp) < 1e-15
    o.step(4)
    bf.step(4)
    got, ref = o.read_fields(), bf.fields()
    assert o.stats()["nonconverged"] == 0
    assert rel_linf(got, ref, "E") < 1e-11
    assert rel_linf(got, ref, "H") < 1e-11
    if magnetic:
        assert rel_linf(got, ref, "M") < 1e-13
        assert max(np.max(np.abs(got[n] - f0[n])) for n in ("Mxx", "Myy", "Mzz")) > 0


# ----------------------------------------------------------------------------- A24 fidelity

@pytest.mark.parametrize("cfg,shape", [(5, (16, 16, 16)), (1, (16, 16, 16)), (4, (16, 16, 24))])
def test_increment_form_is_the_papers_algorithm(cfg, shape):
    """DESIGN.md A24: the fp64 increment-form oracle agrees with eqs. 18-21 evaluated exactly as
    printed in 80-bit arithmetic (state held in 80-bit) to well under the 1e-9 parity bar."""
    w = wl.make_config(cfg, shape=shape)
    a = oracle_from_workload(w, "f64")
    b = oracle_from_workload(w, "ld")
    a.step(40)
    b.step(40)
    fa, fb = a.read_fields(), b.read_fields()
    assert rel_linf(fa, fb, "E") < 5e-9
    assert rel_linf(fa, fb, "H") < 5e-9
    assert rel_linf(fa, fb, "M") < 1e-13
    assert a.stats()["iters_total"] == b.stats()["iters_total"]
