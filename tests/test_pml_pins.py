"""Pins of the oracle's open boundary (split-field PML with multiplicative damping, PAPER.md:189,
reading A26 in DESIGN.md), CPU only.  The paper gives no formulas; what it does state, and what
the mathematics fixes:

PM1  PAPER.md:189: "E and H fields are dissipated with < 0.1 % reflection for non-magnetic
     material aligned with the domain boundaries" -- normal incidence on a 12-cell layer, vacuum
     and a lossless dielectric running into the layer; without the layer the wall reflects 100 %.
PM2  a layer with (almost) zero decay rate is the plain scheme: the split update sums to eq. 11 /
     eq. 21 (a dropped or mis-signed curl term would not).
PM3  oblique incidence and corners: a point source radiating in a 2-D box closed by layers on all
     four sides matches the same source in a box so large that nothing returns, to < 0.5 % of the
     peak at probes near the layers and in the corner region.
PM4  conducting and permeable material running into the layer: still absorbing, and the run is
     stable over many crossings (energy never grows).
"""
import math

import numpy as np
import pytest

from oracle import Oracle

C0 = 299792458.0
MU0 = 4e-7 * math.pi
EPS0 = 1 / (MU0 * C0 * C0)


def _column(nx, pml, eps_r=1.0, steps=0, r0=1e-6):
    """1-D column along x (ny = nz = 1, periodic in y, z), right-moving Gaussian pulse in (Ey, Hz)."""
    dx = 1e-3
    dt = 0.5 * dx / C0
    shp = (1, 1, nx)
    o = Oracle(nx, 1, 1, dx, dx, dx, dt, eps_r=np.full(shp, eps_r), bc=(0, 1, 1), enable_llg=False,
               pml=(pml, pml, 0, 0, 0, 0) if pml else None, pml_r0=r0)
    i = np.arange(nx)
    x0, w = 0.35 * nx, 8.0
    v = C0 / math.sqrt(eps_r)
    ey = np.exp(-0.5 * ((i - x0) / w) ** 2)
    # Hz at (i+1/2), integer time: right-moving wave E/H = eta
    hz = np.exp(-0.5 * ((i + 0.5 - x0) / w) ** 2) * math.sqrt(eps_r * EPS0 / MU0)
    o.set_fields([None, ey.reshape(shp), None], [None, None, hz.reshape(shp)])
    o.step(steps)
    return o.read_fields(("Ey",))["Ey"][0, 0], dt, v, dx


@pytest.mark.parametrize("eps_r", [1.0, 4.0])
def test_pm1_normal_incidence_reflection_below_a_tenth_of_a_percent(eps_r):
    nx, pml = 300, 12
    # time for the pulse to reach the right layer, come back and sit in the middle of the box
    dist = (nx - pml - 0.35 * nx) + 0.45 * nx
    _, dt, v, dx = _column(nx, pml, eps_r)
    steps = int(dist * dx / (v * dt))
    ey, *_ = _column(nx, pml, eps_r, steps)
    wall, *_ = _column(nx, 0, eps_r, steps)
    assert np.max(np.abs(wall)) > 0.9                       # the bare PEC wall sends it all back
    assert np.max(np.abs(ey[pml:nx - pml])) < 1e-3
    # and much later nothing has come back or grown
    late, *_ = _column(nx, pml, eps_r, 4 * steps)
    assert np.max(np.abs(late)) < 1e-3


def test_pm2_zero_rate_layer_is_the_plain_scheme():
    rng = np.random.default_rng(2)
    shape = (10, 9, 8)
    shp = shape[::-1]
    d = (1e-3, 1.2e-3, 0.8e-3)
    dt = 0.9 / (C0 * math.sqrt(sum(1 / h ** 2 for h in d)))
    kw = dict(eps_r=1 + rng.random(shp), sigma=0.5 * rng.random(shp), mu_r=1 + rng.random(shp),
              bc=(0, 0, 1), enable_llg=False)
    E = [rng.standard_normal(shp) for _ in range(3)]
    H = [1e-3 * rng.standard_normal(shp) for _ in range(3)]
    a = Oracle(*shape, *d, dt, **kw)
    b = Oracle(*shape, *d, dt, pml=(3, 2, 4, 0, 0, 0), pml_r0=1 - 1e-13, **kw)
    for o in (a, b):
        o.set_fields(E, H)
        o.set_source(2, (0, 0, 0), shape, None, 1e3, 1e9, 0.0, 100 * dt)
        o.step(12)
    fa, fb = a.read_fields(), b.read_fields()
    for n in ("Ex", "Ey", "Ez", "Hx", "Hy", "Hz"):
        s = max(np.max(np.abs(fa[n])), 1e-300)
        assert np.max(np.abs(fa[n] - fb[n])) / s < 1e-9, n
    # a real layer does change the result
    c = Oracle(*shape, *d, dt, pml=(3, 2, 4, 0, 0, 0), **kw)
    c.set_fields(E, H)
    c.step(12)
    assert np.max(np.abs(c.read_fields()["Ex"] - fa["Ex"])) > 1e-3


def test_pm3_oblique_incidence_and_corners_against_a_large_box():
    n, pml, big = 64, 10, 200
    dx = 1e-3
    dt = 0.9 * dx / (C0 * math.sqrt(3.0))
    f0 = C0 / (12 * dx)                   # 12 cells per wavelength
    steps = 150                           # the wave crosses the small box about twice
    tp = 1.0 / f0

    def run(N, p):
        o = Oracle(N, N, 1, dx, dx, dx, dt, bc=(0, 0, 1), enable_llg=False,
                   pml=(p, p, p, p, 0, 0) if p else None)
        c = N // 2
        o.set_source(2, (c, c, 0), (c + 1, c + 1, 1), None, 1.0, f0, 3 * tp, tp)
        o.step(steps)
        return o.read_fields(("Ez",))["Ez"][0]
    small, ref = run(n, pml), run(big, 0)
    off = big // 2 - n // 2
    ref = ref[off:off + n, off:off + n]
    inner = (slice(pml, n - pml), slice(pml, n - pml))
    peak = np.max(np.abs(ref[inner]))
    assert peak > 0
    # c dt steps / dx = 78 cells > 32: the wave has crossed the box; in the big box it met no wall
    assert 0.9 * dx * steps / math.sqrt(3.0) / dx < (big - n) / 2 + n / 2
    err = np.max(np.abs(small[inner] - ref[inner])) / peak
    assert err < 5e-3, err
    # without the layer the small box is full of reflections
    bare = run(n, 0)
    assert np.max(np.abs(bare[inner] - ref[inner])) / peak > 0.2


def test_pm4_lossy_permeable_material_into_the_layer_is_stable_and_absorbing():
    nx, pml = 120, 10
    dx = 1e-3
    dt = 0.5 * dx / C0
    shp = (1, 1, nx)
    eps = np.full(shp, 2.0)
    mu = np.full(shp, 1.5)
    sig = np.full(shp, 2e-3)
    o = Oracle(nx, 1, 1, dx, dx, dx, dt, eps_r=eps, mu_r=mu, sigma=sig, bc=(0, 1, 1),
               enable_llg=False, pml=(pml, pml, 0, 0, 0, 0))
    i = np.arange(nx)
    ey = np.exp(-0.5 * ((i - 60) / 6.0) ** 2)
    o.set_fields([None, ey.reshape(shp), None])
    prev = None
    for _ in range(12):
        o.step(100)
        f = o.read_fields(("Ey", "Hz"))
        w = float(np.sum(2.0 * EPS0 * f["Ey"] ** 2 + 1.5 * MU0 * f["Hz"] ** 2))
        assert np.isfinite(w)
        if prev is not None:
            assert w <= prev * (1 + 1e-12)
        prev = w
    assert prev < 1e-8 * float(np.sum(2.0 * EPS0 * ey ** 2))


def test_pml_argument_checks():
    shp = (4, 4, 4)
    with pytest.raises(ValueError):
        Oracle(4, 4, 4, 1e-3, 1e-3, 1e-3, 1e-12, bc=(1, 0, 0), enable_llg=False, pml=(2, 0, 0, 0, 0, 0))
    with pytest.raises(ValueError):      # magnetic faces inside the layer
        Oracle(4, 4, 4, 1e-3, 1e-3, 1e-3, 1e-12, bc=(0, 0, 0), enable_llg=True, Ms=np.full(shp, 1e5),
               alpha=np.full(shp, 0.1), gamma=np.full(shp, 1.7e11), pml=(1, 0, 0, 0, 0, 0))
