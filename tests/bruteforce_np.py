"""A second, structurally different statement of the coupled step, for pinning the oracle
on tiny grids (DESIGN.md pin P10).

Whole-array numpy in 80-bit ``np.longdouble``: shifted copies instead of per-point reads,
eqs. 18-21 of PAPER.md:170-181 evaluated exactly as printed (b, a, M^r, N(M), H^r) rather than
in the oracle's increment form, the fixed point run to a fixed iteration count, materials
pre-averaged to edge/face arrays.  Nothing here is shared with ``oracle/`` or the CUDA path.
"""
from __future__ import annotations

import numpy as np

LD = np.longdouble
PI = LD("3.14159265358979323846264338327950288")
MU0 = LD(4) * PI * LD("1e-7")
C0 = LD(299792458)
EPS0 = LD(1) / (MU0 * C0 * C0)

AX = {0: 2, 1: 1, 2: 0}  # grid axis d (x,y,z) -> numpy axis of an array shaped (nz, ny, nx)


def shift(a, d, off, periodic):
    """b[c] = a[c + off*e_d]; wraps when periodic, else reads 0 beyond the stored range."""
    if off == 0:
        return a
    ax = AX[d]
    if periodic:
        return np.roll(a, -off, axis=ax)
    b = np.zeros_like(a)
    n = a.shape[ax]
    src = [slice(None)] * 3
    dst = [slice(None)] * 3
    if off > 0:
        src[ax] = slice(off, n)
        dst[ax] = slice(0, n - off)
    else:
        src[ax] = slice(0, n + off)
        dst[ax] = slice(-off, n)
    b[tuple(dst)] = a[tuple(src)]
    return b


class BruteForce:
    def __init__(self, shape_xyz, d, dt, bc, eps_r, sigma, mu_r, Ms, alpha, gamma, enable_llg,
                 h_bias, hk, axis, iters, scheme=0):
        self.n = shape_xyz
        self.d = [LD(v) for v in d]
        self.dt = LD(dt)
        self.per = [bool(b) for b in bc]
        nx, ny, nz = shape_xyz
        self.shp = (nz, ny, nx)
        f = lambda a, dflt: (np.full(self.shp, LD(dflt)) if a is None
                             else np.asarray(a, dtype=np.float64).reshape(self.shp).astype(LD))
        eps_r, sigma, mu_r = f(eps_r, 1), f(sigma, 0), f(mu_r, 1)
        Ms, alpha, gamma = f(Ms, 0), f(alpha, 0), f(gamma, 0)
        idx = np.indices(self.shp)  # [k, j, i]
        self.pos = {0: idx[2], 1: idx[1], 2: idx[0]}
        # masks of updated (non-wall) faces and edges
        self.face_ok, self.edge_ok = [], []
        for dd in range(3):
            ok = np.ones(self.shp, bool)
            if not self.per[dd]:
                ok &= self.pos[dd] > 0
            self.face_ok.append(ok)
            ok = np.ones(self.shp, bool)
            for t in ((dd + 1) % 3, (dd + 2) % 3):
                if not self.per[t]:
                    ok &= self.pos[t] > 0
            self.edge_ok.append(ok)
        # edge and face materials
        self.eps_e, self.sig_e = [], []
        for dd in range(3):
            t1, t2 = (dd + 1) % 3, (dd + 2) % 3
            m4 = lambda a: (a + shift(a, t1, -1, self.per[t1]) + shift(a, t2, -1, self.per[t2])
                            + shift(shift(a, t1, -1, self.per[t1]), t2, -1, self.per[t2])) / 4
            self.eps_e.append(EPS0 * m4(eps_r))
            self.sig_e.append(m4(sigma))
        m2 = lambda a, dd: (a + shift(a, dd, -1, self.per[dd])) / 2
        self.mu_f = [MU0 * m2(mu_r, dd) for dd in range(3)]
        self.Ms_f = [m2(Ms, dd) for dd in range(3)]
        self.al_f = [m2(alpha, dd) for dd in range(3)]
        self.cf = [MU0 * m2(np.abs(gamma), dd) * self.dt / 4 for dd in range(3)]
        self.mag = [(self.Ms_f[dd] > 0) & self.face_ok[dd] & bool(enable_llg) for dd in range(3)]
        self.hb = [LD(v) for v in h_bias]
        self.hk = LD(hk)
        self.u = [LD(v) for v in axis]
        self.iters = iters
        self.scheme = scheme   # 1: first-order scheme, eqs. 6-9, 12-14
        # electron gyromagnetic ratio: negative; gamma_L = gamma / (1 + alpha^2)
        self.gl_f = [-m2(np.abs(gamma), dd) / (1 + m2(alpha, dd) ** 2) for dd in range(3)]
        self.E = [np.zeros(self.shp, LD) for _ in range(3)]
        self.H = [np.zeros(self.shp, LD) for _ in range(3)]
        self.M = [[np.zeros(self.shp, LD) for _ in range(3)] for _ in range(3)]
        self.sources = []
        self.steps = 0

    def set_fields(self, E, H, M_cell):
        g = lambda a: (np.zeros(self.shp, LD) if a is None
                       else np.asarray(a, np.float64).reshape(self.shp).astype(LD))
        for dd in range(3):
            self.E[dd] = np.where(self.edge_ok[dd], g(E[dd]), 0)
            self.H[dd] = np.where(self.face_ok[dd], g(H[dd]), 0)
        Mc = [g(a) for a in M_cell]
        for dd in range(3):
            m = [(Mc[q] + shift(Mc[q], dd, -1, self.per[dd])) / 2 for q in range(3)]
            nrm = np.sqrt(m[0] ** 2 + m[1] ** 2 + m[2] ** 2)
            safe = np.where(nrm > 0, nrm, 1)
            for q in range(3):
                self.M[dd][q] = np.where(self.mag[dd], m[q] * self.Ms_f[dd] / safe, 0)

    def add_source(self, comp, lo, hi, profile, amplitude, f0, t0, tp, kind=0):
        mask = np.ones(self.shp, bool)
        for dd in range(3):
            mask &= (self.pos[dd] >= lo[dd]) & (self.pos[dd] < hi[dd])
        prof = np.zeros(self.shp, LD)
        if profile is None:
            prof[mask] = 1
        else:
            box = (hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0])
            prof[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = np.asarray(profile, np.float64).reshape(box)
        # (kinds 1-3: hard E, soft H, hard H act on the field arrays themselves)
        self.sources.append((comp, prof, LD(amplitude), LD(f0), LD(t0), LD(tp), kind, mask))

    # -- operators ---------------------------------------------------------------------
    def curl_faces(self, E):
        out = []
        for dd in range(3):
            d1, d2 = (dd + 1) % 3, (dd + 2) % 3
            out.append((shift(E[d2], d1, 1, self.per[d1]) - E[d2]) / self.d[d1]
                       - (shift(E[d1], d2, 1, self.per[d2]) - E[d1]) / self.d[d2])
        return out

    def curl_edges(self, H):
        out = []
        for dd in range(3):
            d1, d2 = (dd + 1) % 3, (dd + 2) % 3
            out.append((H[d2] - shift(H[d2], d1, -1, self.per[d1])) / self.d[d1]
                       - (H[d1] - shift(H[d1], d2, -1, self.per[d2])) / self.d[d2])
        return out

    def heff(self, H, M, dd):
        out = []
        for t in range(3):
            if t == dd:
                h = H[dd]
            else:
                a0 = H[t]
                a1 = shift(a0, dd, -1, self.per[dd])
                h = (a0 + a1 + shift(a0, t, 1, self.per[t]) + shift(a1, t, 1, self.per[t])) / 4
            out.append(h + self.hb[t])
        if self.hk != 0:
            Msafe = np.where(self.Ms_f[dd] > 0, self.Ms_f[dd], 1)
            p = self.hk * (M[0] * self.u[0] + M[1] * self.u[1] + M[2] * self.u[2]) / Msafe
            out = [out[t] + p * self.u[t] for t in range(3)]
        return out

    # -- the step ----------------------------------------------------------------------
    def hm_half(self):
        C = self.curl_faces(self.E)
        Hn = [h.copy() for h in self.H]
        Mn = [[m.copy() for m in self.M[dd]] for dd in range(3)]
        Hnon = [np.where(self.face_ok[dd] & ~self.mag[dd],
                         Hn[dd] - (self.dt / 2 / self.mu_f[dd]) * C[dd], 0) for dd in range(3)]
        Hprev, Mprev = Hn, Mn
        if not any(m.any() for m in self.mag):
            self.H = Hnon
            return
        cr = lambda a, b: [a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2],
                           a[0] * b[1] - a[1] * b[0]]
        if self.scheme == 1:
            # eq. 7 / 12 exactly as printed (with the half step dt/2), N(M), then eq. 9 / 14
            Hcur, Mcur = [], []
            for dd in range(3):
                Msf = np.where(self.mag[dd], self.Ms_f[dd], 1)
                hn = self.heff(Hn, Mn[dd], dd)
                mxh = cr(Mn[dd], hn)
                mxmxh = cr(Mn[dd], mxh)
                g = MU0 * self.gl_f[dd]
                m = [Mn[dd][q] + (self.dt / 2) * (g * mxh[q] + self.al_f[dd] * g / Msf * mxmxh[q])
                     for q in range(3)]
                nrm = np.sqrt(m[0] ** 2 + m[1] ** 2 + m[2] ** 2)
                nrm = np.where(self.mag[dd], nrm, 1)
                m = [np.where(self.mag[dd], m[q] * Msf / nrm, 0) for q in range(3)]
                h = Hn[dd] + Mn[dd][dd] - m[dd] - (self.dt / 2 / MU0) * C[dd]
                Hcur.append(np.where(self.mag[dd], h, Hnon[dd]))
                Mcur.append(m)
            self.H, self.M = Hcur, Mcur
            return
        for _ in range(self.iters):
            Hcur, Mcur = [], []
            for dd in range(3):
                Msf = np.where(self.mag[dd], self.Ms_f[dd], 1)
                hn = self.heff(Hn, Mn[dd], dd)
                he = self.heff(Hprev, Mprev[dd], dd)
                x = cr(Mn[dd], hn)
                b = [Mn[dd][q] - self.cf[dd] * x[q] for q in range(3)]                  # (20)
                a = [-(self.cf[dd] * he[q] + self.al_f[dd] / Msf * Mn[dd][q]) for q in range(3)]  # (19)
                ab = a[0] * b[0] + a[1] * b[1] + a[2] * b[2]
                axb = cr(a, b)
                den = 1 + a[0] ** 2 + a[1] ** 2 + a[2] ** 2
                m = [(b[q] + ab * a[q] - axb[q]) / den for q in range(3)]               # (18)
                nrm = np.sqrt(m[0] ** 2 + m[1] ** 2 + m[2] ** 2)
                nrm = np.where(self.mag[dd], nrm, 1)
                m = [np.where(self.mag[dd], m[q] * Msf / nrm, 0) for q in range(3)]     # N(M)
                h = Hn[dd] + Mn[dd][dd] - m[dd] - (self.dt / 2 / MU0) * C[dd]           # (21)
                Hcur.append(np.where(self.mag[dd], h, Hnon[dd]))
                Mcur.append(m)
            Hprev, Mprev = Hcur, Mcur
        self.H, self.M = Hprev, Mprev

    def e_update(self):
        t = (LD(self.steps) + LD(0.5)) * self.dt
        cH = self.curl_edges(self.H)
        for dd in range(3):
            J = np.zeros(self.shp, LD)
            for comp, prof, A, f0, t0, tp, kind, _ in self.sources:
                if comp == dd and kind == 0:
                    J = J + A * np.exp(-((t - t0) ** 2) / (2 * tp * tp)) * np.cos(2 * PI * f0 * t) * prof
            s, e = self.sig_e[dd], self.eps_e[dd]
            new = (cH[dd] - (s / 2 - e / self.dt) * self.E[dd] - J) / (s / 2 + e / self.dt)   # (11)
            self.E[dd] = np.where(self.edge_ok[dd], new, 0)

    def field_sources(self, kind, t):
        for comp, prof, A, f0, t0, tp, knd, mask in self.sources:
            if knd != kind:
                continue
            v = A * np.exp(-((t - t0) ** 2) / (2 * tp * tp)) * np.cos(2 * PI * f0 * t) * prof
            if kind == 1:
                m = mask & self.edge_ok[comp]
                self.E[comp] = np.where(m, v, self.E[comp])
            else:
                m = mask & self.face_ok[comp]
                self.H[comp] = np.where(m, self.H[comp] + self.dt * v if kind == 2 else v, self.H[comp])

    def step(self, n=1):
        for _ in range(n):
            self.field_sources(2, LD(self.steps) * self.dt)          # soft H: start of the step
            self.hm_half()
            self.e_update()
            self.field_sources(1, LD(self.steps + 1) * self.dt)      # hard E: after its update
            self.hm_half()
            self.field_sources(3, LD(self.steps + 1) * self.dt)      # hard H: after its update
            self.steps += 1

    def fields(self):
        out = {}
        for dd, c in enumerate("xyz"):
            out["E" + c] = self.E[dd].astype(np.float64)
            out["H" + c] = self.H[dd].astype(np.float64)
            for q, cc in enumerate("xyz"):
                out["M" + c + cc] = self.M[dd][q].astype(np.float64)
        return out
