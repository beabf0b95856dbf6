"""Seeded synthetic inputs for the coupled FDTD-LLG path (the five BASELINE.json configs).

This module serves BOTH the oracle-side tests and the CUDA path, and therefore holds none of
the method's arithmetic: it only builds grids, material maps, initial fields and source
descriptions.  Every random number comes from a counter-based generator (splitmix64 of
seed/stream/cell-index), so any sub-box of any array can be generated independently, on the
host or on the GPU (all tensor code is plain ``torch`` ops and runs on either device).

Recipes: the paper's workloads are its own waveguide and
tunable-filter geometries; no public dataset is involved.  The five
configs are synthetic stand-ins with those shapes -- long guide axis, thin magnetic slab in a
mostly non-magnetic box, PEC walls -- at dx = 1 um and 0.9 x the vacuum Courant step.
Reduced shapes (``shape=``) keep every geometric feature at the same FRACTION of the box, so
that a small grid the oracle finishes in seconds has the structure of the full one.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import torch

MU0 = 4.0e-7 * math.pi
C0 = 299792458.0
EPS0 = 1.0 / (MU0 * C0 * C0)
ETA0 = math.sqrt(MU0 / EPS0)

_MASK64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
BASE_SEED = 210312819

PEC, PERIODIC = 0, 1


# ----------------------------------------------------------------------------- generator

def _s64(x: int) -> int:
    """Two's-complement int64 view of an unsigned 64-bit constant."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of an int64 tensor holding uint64 bit patterns."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def splitmix64_py(seed: int, stream: int, idx: int) -> int:
    """Pure-python reference of the generator (tests pin the tensor code to this)."""
    z = (seed + _GOLDEN * ((stream << 40) + idx + 1)) & _MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
    return z ^ (z >> 31)


def uniform(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """u in [0,1): u = (splitmix64(seed + G*(stream*2^40 + idx + 1)) >> 11) * 2^-53."""
    z = (idx + ((stream << 40) + 1)) * _s64(_GOLDEN) + _s64(seed)
    z = (z ^ _lsr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _s64(0x94D049BB133111EB)
    z = z ^ _lsr(z, 31)
    return _lsr(z, 11).to(torch.float64) * (2.0 ** -53)


def normal(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """Standard normal by Box-Muller on streams (2*stream, 2*stream+1)."""
    u1 = uniform(seed, 2 * stream, idx)
    u2 = uniform(seed, 2 * stream + 1, idx)
    return torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos(2.0 * math.pi * u2)


def courant_dt(cfl: float, dx: float, dy: float, dz: float) -> float:
    """cfl x the vacuum Courant limit."""
    return cfl / (C0 * math.sqrt(1.0 / dx ** 2 + 1.0 / dy ** 2 + 1.0 / dz ** 2))


def yee_omega_dt(kvec, d, dt) -> float:
    """omega*dt of the Yee scheme for wave vector kvec: sin^2(w dt/2) = (c dt)^2 sum sin^2(k_a d_a/2)/d_a^2."""
    s = sum((math.sin(0.5 * k * h) / h) ** 2 for k, h in zip(kvec, d))
    return 2.0 * math.asin(C0 * dt * math.sqrt(s))


# ----------------------------------------------------------------------------- container

@dataclass
class Source:
    comp: int
    lo: tuple
    hi: tuple
    amplitude: float
    f0: float
    t0: float
    tp: float
    profile: Optional[torch.Tensor] = None
    kind: int = 0   # 0 soft E (J of eq. 11), 1 hard E, 2 soft H, 3 hard H


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    dt: float
    bc: tuple
    steps: int
    enable_llg: bool = False
    h_bias: tuple = (0.0, 0.0, 0.0)
    ani_hk: float = 0.0
    ani_axis: tuple = (0.0, 0.0, 1.0)
    llg_tol: float = 1e-12
    llg_max_iter: int = 20
    # cell-centred material maps, shape (nz, ny, nx) float64; a python float = uniform value;
    # missing/None = the default
    materials: dict = field(default_factory=dict)
    E: list = field(default_factory=lambda: [None, None, None])
    H: list = field(default_factory=lambda: [None, None, None])
    M_cell: list = field(default_factory=lambda: [None, None, None])
    sources: list = field(default_factory=list)
    pml: Optional[tuple] = None     # (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi) cells of the open boundary layer
    pml_r0: Optional[float] = None
    pml_order: Optional[int] = None
    slab_ext: tuple = (0, 0)        # this workload is one z-slab of a larger grid: its arrays carry the
                                    # neighbours' adjacent plane on the flagged sides (slabs.cut_workload)
    seed: int = BASE_SEED
    notes: str = ""

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    def numpy(self):
        """Host numpy views of every array (for the oracle)."""
        import numpy as np

        def cv(t):
            if t is None:
                return None
            if isinstance(t, (int, float)):   # uniform material given as a scalar
                return np.full((self.nz + sum(self.slab_ext), self.ny, self.nx), float(t))
            return t.detach().cpu().numpy()
        return {
            "materials": {k: cv(v) for k, v in self.materials.items()},
            "E": [cv(t) for t in self.E],
            "H": [cv(t) for t in self.H],
            "M_cell": [cv(t) for t in self.M_cell],
        }


def _grid(nx, ny, nz, device, k0=0, k1=None):
    """Index tensors i (1,1,nx), j (1,ny,1), k (nk,1,1) and the flat cell index."""
    k1 = nz if k1 is None else k1
    i = torch.arange(nx, device=device, dtype=torch.int64).view(1, 1, nx)
    j = torch.arange(ny, device=device, dtype=torch.int64).view(1, ny, 1)
    k = torch.arange(k0, k1, device=device, dtype=torch.int64).view(k1 - k0, 1, 1)
    return i, j, k, i + nx * (j + ny * k)


def _slabs(nz, planes=16):
    for k0 in range(0, nz, planes):
        yield k0, min(nz, k0 + planes)


def _zeros(nx, ny, nz, device):
    return torch.zeros((nz, ny, nx), dtype=torch.float64, device=device)


def tilted_m_cell(seed, nx, ny, nz, Ms, theta_max_deg, device, stream0=20):
    """M_cell = Ms (sin t cos p, sin t sin p, cos t), t = theta_max*u1, p = 2 pi u2, per cell.
    ``Ms`` is the (nz,ny,nx) saturation map (zero outside the magnet)."""
    out = [_zeros(nx, ny, nz, device) for _ in range(3)]
    tmax = math.radians(theta_max_deg)
    for k0, k1 in _slabs(nz):
        _, _, _, idx = _grid(nx, ny, nz, device, k0, k1)
        th = tmax * uniform(seed, stream0, idx)
        ph = 2.0 * math.pi * uniform(seed, stream0 + 1, idx)
        ms = Ms[k0:k1]
        st = torch.sin(th)
        out[0][k0:k1] = ms * st * torch.cos(ph)
        out[1][k0:k1] = ms * st * torch.sin(ph)
        out[2][k0:k1] = ms * torch.cos(th)
    return out


# ----------------------------------------------------------------------------- the configs

def config1(shape=(32, 32, 32), device="cpu", steps=100) -> Workload:
    """All-magnetic PEC box, Gaussian Ex pulse (BASELINE.json configs[0])."""
    nx, ny, nz = shape
    seed = BASE_SEED + 1
    dx = 1e-6
    w = Workload("cfg1_pec_allmagnetic", nx, ny, nz, dx, dx, dx, courant_dt(0.9, dx, dx, dx),
                 (PEC, PEC, PEC), steps, enable_llg=True, h_bias=(0.0, 0.0, 1e4),
                 llg_tol=1e-12, llg_max_iter=20, seed=seed)
    Ms = torch.full((nz, ny, nx), 1.4e5, dtype=torch.float64, device=device)
    w.materials = {"Ms": Ms,
                   "alpha": torch.full_like(Ms, 0.005),
                   "gamma": torch.full_like(Ms, 1.759e11)}
    w.M_cell = tilted_m_cell(seed, nx, ny, nz, Ms, 1.0, device)
    jit = [4.0 * float(uniform(seed, 10, torch.tensor([q]))[0]) - 2.0 for q in range(3)]
    i, j, k, _ = _grid(nx, ny, nz, device)
    sig = 4.0 * min(nx, ny, nz) / 32.0
    r2 = ((i + 0.5 - (nx / 2 + jit[0])) ** 2 + (j - (ny / 2 + jit[1])) ** 2
          + (k - (nz / 2 + jit[2])) ** 2).to(torch.float64)
    w.E[0] = 1e6 * torch.exp(-r2 / (2.0 * sig * sig))
    return w


def config2(shape=(256, 256, 256), device="cpu", steps=1000, noise=1e-6, wavelength_cells=32
            ) -> Workload:
    """Vacuum, periodic, exact Yee eigenmode along x (Ey/Hz) + seeded noise (configs[1]).
    H amplitude is cos(w dt/2)/eta0 and H sits half a cell further: the scheme's integer-time
    H is the mean of the leapfrog H^{n+-1/2} (DESIGN.md pin P1)."""
    nx, ny, nz = shape
    seed = BASE_SEED + 2
    dx = 1e-6
    dt = courant_dt(0.9, dx, dx, dx)
    w = Workload("cfg2_vacuum_periodic", nx, ny, nz, dx, dx, dx, dt,
                 (PERIODIC, PERIODIC, PERIODIC), steps, enable_llg=False, seed=seed)
    kx = 2.0 * math.pi / (wavelength_cells * dx)
    wdt = yee_omega_dt((kx, 0.0, 0.0), (dx, dx, dx), dt)
    for c in range(3):
        w.E[c] = _zeros(nx, ny, nz, device)
        w.H[c] = _zeros(nx, ny, nz, device)
    for k0, k1 in _slabs(nz):
        i, _, _, idx = _grid(nx, ny, nz, device, k0, k1)
        for c in range(3):
            if noise:
                w.E[c][k0:k1] = noise * (2.0 * uniform(seed, 30 + c, idx) - 1.0)
                w.H[c][k0:k1] = (noise / ETA0) * (2.0 * uniform(seed, 33 + c, idx) - 1.0)
        w.E[1][k0:k1] += torch.cos(kx * dx * i.to(torch.float64))
        w.H[2][k0:k1] += (math.cos(0.5 * wdt) / ETA0) * torch.cos(kx * dx * (i.to(torch.float64) + 0.5))
    w.notes = f"omega*dt={wdt!r} kx*dx={kx * dx!r}"
    return w


def bandwidth_tp(f0: float, frac_bw: float) -> float:
    """T_p of eq. 31's Gaussian envelope whose spectral FWHM is frac_bw*f0 (A15)."""
    return 2.0 * math.sqrt(2.0 * math.log(2.0)) / (2.0 * math.pi * frac_bw * f0)


def config3(shape=(512, 128, 128), device="cpu", steps=2000) -> Workload:
    """Waveguide-like: PEC box, dielectric slab, two conductor strips, soft Jy source (configs[2])."""
    nx, ny, nz = shape
    seed = BASE_SEED + 3
    dx = 1e-6
    w = Workload("cfg3_waveguide", nx, ny, nz, dx, dx, dx, courant_dt(0.9, dx, dx, dx),
                 (PEC, PEC, PEC), steps, enable_llg=False, seed=seed)
    eps = torch.ones((nz, ny, nx), dtype=torch.float64, device=device)
    sig = torch.zeros_like(eps)
    kslab = max(1, nz // 8)                      # 16 of 128
    eps[:kslab] = 11.7
    sw = max(1, ny // 16)                        # 8 of 128
    j1, j2 = (ny * 44) // 128, (ny * 76) // 128  # 44 and 76 of 128
    kt = min(nz, kslab + 2)                      # 2 cells thick
    sig[kslab:kt, j1:j1 + sw, :] = 5.8e7
    sig[kslab:kt, j2:j2 + sw, :] = 5.8e7
    w.materials = {"eps_r": eps, "sigma": sig}
    f0 = 10e9
    tp = bandwidth_tp(f0, 0.4)
    isrc = min(nx - 1, max(1, nx // 64))         # 8 of 512
    w.sources = [Source(1, (isrc, 0, 0), (isrc + 1, ny, nz), 1e9, f0, 3.0 * tp, tp)]
    return w


def config4(shape=(384, 384, 384), device="cpu", steps=2000) -> Workload:
    """Tunable-filter-like: PEC box, thin magnetic slab with uniaxial anisotropy, Jx source (configs[3])."""
    nx, ny, nz = shape
    seed = BASE_SEED + 4
    dx = 1e-6
    w = Workload("cfg4_tunable_filter", nx, ny, nz, dx, dx, dx, courant_dt(0.9, dx, dx, dx),
                 (PEC, PEC, PEC), steps, enable_llg=True, h_bias=(0.0, 0.0, 8e4), ani_hk=2e3,
                 ani_axis=(0.0, 0.0, 1.0), llg_tol=1e-12, llg_max_iter=20, seed=seed)
    kslab = max(1, nz // 12)                     # 32 of 384
    Ms = _zeros(nx, ny, nz, device)
    Ms[:kslab] = 1.4e5
    w.materials = {"Ms": Ms, "alpha": 1e-3, "gamma": 1.759e11}
    w.M_cell = tilted_m_cell(seed, nx, ny, nz, Ms, 0.5, device)
    f0 = 5e9
    tp = 1.0 / f0
    ks = min(nz - 1, max(kslab + 1, nz // 8))    # 48 of 384
    w.sources = [Source(0, (0, 0, ks), (nx, ny, ks + 1), 1e9, f0, 3.0 * tp, tp)]
    return w


def config5(shape=(768, 768, 768), device="cpu", steps=200, e_fields=True) -> Workload:
    """Large coupled grid: periodic x,y / PEC z, lower half magnetic, E ~ N(0,1) V/m (configs[4])."""
    nx, ny, nz = shape
    seed = BASE_SEED + 5
    dx = 1e-6
    w = Workload("cfg5_large_coupled", nx, ny, nz, dx, dx, dx, courant_dt(0.9, dx, dx, dx),
                 (PERIODIC, PERIODIC, PEC), steps, enable_llg=True, h_bias=(0.0, 0.0, 5e4),
                 llg_tol=1e-12, llg_max_iter=20, seed=seed)
    Ms = _zeros(nx, ny, nz, device)
    Ms[: nz // 2] = 8e5
    w.materials = {"Ms": Ms, "alpha": 0.01, "gamma": 1.759e11}
    w.M_cell = tilted_m_cell(seed, nx, ny, nz, Ms, 2.0, device)
    if e_fields:
        for c in range(3):
            w.E[c] = _zeros(nx, ny, nz, device)
            for k0, k1 in _slabs(nz):
                _, _, _, idx = _grid(nx, ny, nz, device, k0, k1)
                w.E[c][k0:k1] = normal(seed, 40 + c, idx)
    return w


def paper_convergence_test(n: int, steps: int, device="cpu") -> Workload:
    """The paper's own convergence test (eqs. 22-28), not a BASELINE config:
    fully periodic cube of side L = 0.1 m centred at the origin on an n^3 grid, plane-wave-like
    E, H (eqs. 22-23, sampled at the Yee locations), Gaussian bumps of sigma, eps, Ms, alpha,
    gamma around the origin (eqs. 24-28, sampled at cell centres), M = (Ms, 0, 0), no bias,
    CFL 0.9 on the vacuum speed of light, the paper's tolerance 1e-6."""
    L = 0.1
    h = L / n
    w = Workload(f"paper_convergence_{n}", n, n, n, h, h, h, courant_dt(0.9, h, h, h),
                 (PERIODIC, PERIODIC, PERIODIC), steps, enable_llg=True, llg_tol=1e-6,
                 llg_max_iter=50)
    idx = torch.arange(n, device=device, dtype=torch.float64)
    cen = -L / 2 + (idx + 0.5) * h      # cell centres / face and edge mid-points
    nod = -L / 2 + idx * h              # nodes
    ax = lambda v, a: v.view([n if q == a else 1 for q in range(3)]).expand(n, n, n).contiguous()
    # tensor axes: 0 = z, 1 = y, 2 = x
    r2 = ax(cen, 0) ** 2 + ax(cen, 1) ** 2 + ax(cen, 2) ** 2
    g = torch.exp(-1000.0 * r2)
    w.materials = {"eps_r": 1.0 + g, "sigma": 0.1 * g, "Ms": 1e4 * (1.0 + g),
                   "alpha": 0.5 * (1.0 + g), "gamma": -1.759e11 * (1.0 + g)}
    k20 = 20.0 * math.pi
    a0 = 1e6
    w.E = [a0 * torch.cos(k20 * ax(nod, 0)),    # Ex(z) on the x-edge (i+1/2, j, k): z is a node
           a0 * torch.cos(k20 * ax(nod, 2)),    # Ey(x) on (i, j+1/2, k)
           a0 * torch.cos(k20 * ax(nod, 1))]    # Ez(y) on (i, j, k+1/2)
    b0 = a0 / (120.0 * math.pi)
    w.H = [b0 * torch.cos(k20 * ax(cen, 1)),    # Hx(y) on the x-face (i, j+1/2, k+1/2)
           b0 * torch.cos(k20 * ax(cen, 0)),    # Hy(z) on (i+1/2, j, k+1/2)
           b0 * torch.cos(k20 * ax(cen, 2))]    # Hz(x) on (i+1/2, j+1/2, k)
    w.M_cell = [w.materials["Ms"].clone(), None, None]
    return w


def paper_air_waveguide(nx=512, ny=4, nz=512, npml=16, device="cpu") -> Workload:
    """The paper's first validation device (Fig. 4a): air-filled X-band
    rectangular waveguide, W = 14.95 mm (x), h = 10.16 mm (y), 500 mm long (z) on 512 x 4 x 512
    cells, CFL 0.8; PEC side walls and PEC at z = +L/2 where a surface current "directly added on
    top of the H field" launches the TE10 mode towards -z (eq. 31: f0 = 10.5 GHz, T_p one period,
    centred at 3 T_p).  Readings: the excitation is a HARD source on the tangential Hx faces next to
    the wall, H_x = I(t) cos(pi x / W) with x measured from the guide axis (the TE10 profile; the
    printed shape function cos(2 pi x / (W/2)) is not that mode: taken as garbled); the far end is
    closed by the open boundary (npml cells)."""
    W, h, L = 14.95e-3, 10.16e-3, 500e-3
    dx, dy, dz = W / nx, h / ny, L / nz
    w = Workload("paper_air_waveguide", nx, ny, nz, dx, dy, dz, courant_dt(0.8, dx, dy, dz),
                 (PEC, PEC, PEC), 80000, enable_llg=False)
    w.pml = (0, 0, 0, 0, npml, 0)
    f0 = 10.5e9
    tp = 1.0 / f0
    x = -W / 2 + torch.arange(nx, device=device, dtype=torch.float64) * dx     # Hx faces sit at x_i
    prof = torch.cos(math.pi * x / W).view(1, 1, nx).expand(1, ny, nx).contiguous()
    w.sources = [Source(0, (0, 0, nz - 1), (nx, ny, nz), 1.0, f0, 3.0 * tp, tp, prof, 3)]
    return w


def paper_tunable_filter(nx=1024, ny=4, nz=512, npml=16, device="cpu") -> Workload:
    """The paper's second validation device (Fig. 4b): the waveguide of
    `paper_air_waveguide` with a YIG slab 0.45 mm thick along z, one face on a side wall:
    4 pi Ms = 1750 G (Ms = 1.3926e5 A/m), alpha = 0.0051, eps_r = 13, bias H0 = 2890 Oe
    (2.2998e5 A/m) along y, M saturated along the bias; 1024 x 4 x 512 cells, CFL
    0.8, the paper's tolerance 1e-6.  Readings as `paper_air_waveguide`; in addition the slab sits on
    the x = -W/2 wall and stops two cells short of the open-boundary layer (no magnetic cell may
    touch it)."""
    W, h, L = 14.95e-3, 10.16e-3, 500e-3
    dx, dy, dz = W / nx, h / ny, L / nz
    w = Workload("paper_tunable_filter", nx, ny, nz, dx, dy, dz, courant_dt(0.8, dx, dy, dz),
                 (PEC, PEC, PEC), 80000, enable_llg=True, h_bias=(0.0, 2.2998e5, 0.0),
                 llg_tol=1e-6, llg_max_iter=20)
    w.pml = (0, 0, 0, 0, npml, 0)
    ncell = max(1, int(round(0.45e-3 / dx)))
    Ms = _zeros(nx, ny, nz, device)
    eps = torch.ones((nz, ny, nx), dtype=torch.float64, device=device)
    k0 = npml + 2
    Ms[k0:, :, :ncell] = 1.3926e5
    eps[k0:, :, :ncell] = 13.0
    w.materials = {"Ms": Ms, "alpha": 0.0051, "gamma": 1.759e11, "eps_r": eps}
    w.M_cell = [None, Ms.clone(), None]
    f0 = 10.5e9
    tp = 1.0 / f0
    x = -W / 2 + torch.arange(nx, device=device, dtype=torch.float64) * dx
    prof = torch.cos(math.pi * x / W).view(1, 1, nx).expand(1, ny, nx).contiguous()
    w.sources = [Source(0, (0, 0, nz - 1), (nx, ny, nz), 1.0, f0, 3.0 * tp, tp, prof, 3)]
    return w


def config6(shape=(1024, 4, 512), device="cpu", steps=80000) -> Workload:
    """Not a BASELINE.json config: the paper's own weak-scaling base case (the
    tunable filter on 1024 x 4 x 512 cells per GPU), for `bench.py --config 6`."""
    w = paper_tunable_filter(shape[0], shape[1], shape[2], device=device)
    w.steps = steps
    return w


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5, 6: config6}

# shapes the oracle finishes in seconds: several tiles of the kernels plus a ragged tail
SMALL_SHAPES = {1: (32, 32, 32), 2: (40, 36, 28), 3: (72, 40, 36), 4: (44, 36, 40),
                5: (40, 44, 36)}


def make_config(n: int, shape=None, device="cpu", steps=None, **kw) -> Workload:
    f = CONFIGS[n]
    args = dict(device=device, **kw)
    if shape is not None:
        args["shape"] = tuple(shape)
    if steps is not None:
        args["steps"] = steps
    return f(**args)
