"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: it only evaluates closed-form initial fields.  The paper's own workloads are MESA-derived
stellar models that are not available; these stand in for them with the same shape:
Mach ~0.035 (L25), concentrations down to 1e-5 (L25), a spherical convection zone under a stable layer
inside a cube with gravity tapered to zero before the wall (L69), fp32 state (L35).

Every field is a pure function of the GLOBAL cell index and a handful of numbers drawn from
numpy.default_rng(181013416 + cfg); it is evaluated in fp64 and rounded once to fp32, so any sub-box
(window) can be regenerated exactly.  torch is used only as an array library (CPU or CUDA device).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

BC_PERIODIC, BC_REFLECT = 0, 1
GRAV_NONE, GRAV_CONST_Z, GRAV_RADIAL = 0, 1, 2
NF = 15
NG = 4
SEED0 = 181013416
GAMMA = 5.0 / 3.0

# Legendre basis on [-1/2, 1/2]: P0 = 1, P1 = s, P2 = s^2 - 1/12, norms 1, 1/12, 1/180.
# Coefficient order m000 m100 m010 m001 m200 m020 m002 m110 m101 m011 (exponents along x, y, z).
_ABC = ((0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (0, 2, 0), (0, 0, 2), (1, 1, 0), (1, 0, 1), (0, 1, 1))
_NORM = (1.0, 1.0 / 12.0, 1.0 / 180.0)
_GL_X = (-0.5 * math.sqrt(3.0 / 5.0), 0.0, 0.5 * math.sqrt(3.0 / 5.0))
_GL_W = (5.0 / 18.0, 8.0 / 18.0, 5.0 / 18.0)


def _P(n, s):
    return 1.0 if n == 0 else (s if n == 1 else s * s - 1.0 / 12.0)


def _modes(rng, K, kmax, dims=3):
    """K plane waves: integer wave vectors in [-kmax, kmax]^dims (not all zero), phases, amplitudes."""
    ks = []
    while len(ks) < K:
        k = rng.integers(-kmax, kmax + 1, size=dims)
        if np.any(k != 0):
            ks.append(k)
    ks = np.array(ks, dtype=np.float64)
    phi = rng.uniform(0.0, 2.0 * math.pi, size=K)
    amp = rng.uniform(0.5, 1.0, size=K)
    return ks, phi, amp


def _eval_modes(modes, coords, rms):
    """sum_m A_m sin(2 pi k_m.x + phi_m), rescaled by the analytic rms sqrt(sum A^2 / 2) to `rms`."""
    ks, phi, amp = modes
    scale = rms / math.sqrt(float(np.sum(amp * amp)) / 2.0)
    out = None
    for m in range(len(phi)):
        ph = None
        for d, x in enumerate(coords):
            t = (2.0 * math.pi * float(ks[m, d])) * x
            ph = t if ph is None else ph + t
        term = (scale * float(amp[m])) * torch.sin(ph + float(phi[m]))
        out = term if out is None else out + term
    return out


@dataclass
class Workload:
    cfg: int
    name: str
    n: int                      # cells per side
    steps: int
    cfl: float
    bc: tuple                   # xlo xhi ylo yhi zlo zhi
    grav: dict | None           # kind, s0, ds, center, g, rho0, p0 (fp32 numpy) or None
    gamma: float = GAMMA
    rho_floor: float = 1e-10
    p_floor: float = 1e-10
    _p: dict = field(default_factory=dict, repr=False)

    @property
    def dx(self):
        return 1.0 / self.n

    @property
    def shape(self):
        return (self.n, self.n, self.n)

    # -------------------------------------------------------------------------------------------
    def _coords(self, lo, hi, device, off=(0.0, 0.0, 0.0)):
        """broadcastable fp64 cell-centre coordinates x [1,1,nx], y [1,ny,1], z [nz,1,1] (+ offset in cells)."""
        dx = self.dx
        mk = lambda a, b, o: (torch.arange(a, b, device=device, dtype=torch.float64) + (0.5 + o)) * dx
        x = mk(lo[0], hi[0], off[0]).view(1, 1, -1)
        y = mk(lo[1], hi[1], off[1]).view(1, -1, 1)
        z = mk(lo[2], hi[2], off[2]).view(-1, 1, 1)
        return x, y, z

    def _table_interp(self, name, s):
        """linear interpolation of the fp32 gravity-table column `name` at fp64 positions s."""
        g = self.grav
        tab = torch.as_tensor(np.asarray(g[name], dtype=np.float64), device=s.device)
        t = (s - g["s0"]) / g["ds"]
        k = torch.clamp(torch.floor(t), 0, tab.numel() - 2)
        w = t - k
        k = k.long()
        return (1.0 - w) * tab[k] + w * tab[k + 1]

    def _fv(self, x, y, z):
        raise NotImplementedError

    def _hydro(self, x, y, z):
        raise NotImplementedError

    def fields(self, lo=(0, 0, 0), hi=None, device="cpu"):
        """Full-state fp32 fields [15][nz][ny][nx] of the sub-box with global index range [lo, hi)."""
        hi = tuple(hi) if hi is not None else self.shape
        lo = tuple(lo)
        assert all(0 <= a < b <= self.n for a, b in zip(lo, hi))
        shp = (hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0])
        out = torch.empty((NF,) + shp, dtype=torch.float32, device=device)
        x, y, z = self._coords(lo, hi, device)
        for f, v in enumerate(self._hydro(x, y, z)):
            out[f] = v.expand(shp).to(torch.float32) if torch.is_tensor(v) else float(v)
        # PPB coefficients: 3x3x3 Gauss-Legendre projection of the FV formula onto the Legendre basis
        acc = [torch.zeros(shp, dtype=torch.float64, device=device) for _ in range(10)]
        for a in range(3):
            for b in range(3):
                for c in range(3):
                    xs, ys, zs = self._coords(lo, hi, device, off=(_GL_X[a], _GL_X[b], _GL_X[c]))
                    wv = (_GL_W[a] * _GL_W[b] * _GL_W[c]) * self._fv(xs, ys, zs)
                    for k, (ea, eb, ec) in enumerate(_ABC):
                        pw = _P(ea, _GL_X[a]) * _P(eb, _GL_X[b]) * _P(ec, _GL_X[c])
                        if pw != 0.0:
                            acc[k] += pw * wv
        for k, (ea, eb, ec) in enumerate(_ABC):
            out[5 + k] = (acc[k] / (_NORM[ea] * _NORM[eb] * _NORM[ec])).to(torch.float32)
        return out


# ------------------------------------------------------------------------------------------------
class _Cfg1(Workload):
    """32^3 periodic cube, g = 0: rho = 1 + 0.1 sum_3 sin, p = 0.6 (c = 1), velocity rms 0.035, FV tanh slab in z."""

    def _hydro(self, x, y, z):
        p = self._p
        ks, phi, _ = p["rho_modes"]
        rho = 1.0
        for m in range(3):
            rho = rho + 0.1 * torch.sin(2.0 * math.pi * (float(ks[m, 0]) * x + float(ks[m, 1]) * y + float(ks[m, 2]) * z)
                                        + float(phi[m]))
        vr = 0.035 / math.sqrt(3.0)
        u = [_eval_modes(p["vel_modes"][d], (x, y, z), vr) for d in range(3)]
        return rho, u[0], u[1], u[2], 0.6

    def _fv(self, x, y, z):
        return (0.5 + 0.4 * torch.tanh((0.25 - torch.abs(z - 0.5)) / (2.0 * self.dx))) + 0.0 * (x + y)


class _Cfg2(Workload):
    """Stratified box, constant gravity -z, isentropic lower half / isothermal upper half, reflecting z walls."""

    @staticmethod
    def base(z):
        """closed-form hydrostatic base state (numpy fp64): enthalpy 1.5 - z below z = 0.5, isothermal above."""
        z = np.asarray(z, dtype=np.float64)
        h = 1.5 - np.minimum(z, 0.5)
        rho_lo = (h / 1.5) ** 1.5
        p_lo = 0.6 * rho_lo ** GAMMA
        rho_t = (1.0 / 1.5) ** 1.5
        p_t = 0.6 * rho_t ** GAMMA
        H = p_t / rho_t
        e = np.exp(-np.maximum(z - 0.5, 0.0) / H)
        return np.where(z < 0.5, rho_lo, rho_t * e), np.where(z < 0.5, p_lo, p_t * e)

    def _hydro(self, x, y, z):
        p = self._p
        # zero perturbation: the field IS the fp32 table node at the cell centre (node 2k + 9)
        kz = torch.round(z / self.dx - 0.5).long().view(-1)
        r0 = torch.as_tensor(np.asarray(self.grav["rho0"], dtype=np.float64), device=z.device)[2 * kz + 2 * NG + 1]
        p0 = torch.as_tensor(np.asarray(self.grav["p0"], dtype=np.float64), device=z.device)[2 * kz + 2 * NG + 1]
        u = [_eval_modes(p["vel_modes"][d], (x, y, z), 1e-3) for d in range(3)]
        u[2] = u[2] * torch.sin(math.pi * z)
        return r0.view(-1, 1, 1), u[0], u[1], u[2], p0.view(-1, 1, 1)

    def _fv(self, x, y, z):
        return 0.5 * (1.0 + torch.tanh((z - 0.6) / self.dx)) + 0.0 * (x + y)


class _Cfg3(Workload):
    """Blast in stratified gas: density contrast 1000 across a perturbed tanh interface, 1e4 pressure spike."""

    def _zi(self, x, y):
        return 0.5 + 0.01 * _eval_modes(self._p["if_modes"], (x, y), 1.0)

    def _hydro(self, x, y, z):
        dx = self.dx
        zi = self._zi(x, y)
        rho = 1.0 + 999.0 * 0.5 * (1.0 - torch.tanh((z - zi) / (2.0 * dx)))
        d2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
        pr = 1.0 + (1.0e4 - 1.0) * torch.exp(-d2 / (8.0 * dx) ** 2)
        return rho, 0.0, 0.0, 0.0, pr

    def _fv(self, x, y, z):
        return 1.0e-5 * 0.5 * (1.0 - torch.tanh((z - self._zi(x, y)) / (2.0 * self.dx)))


class _Cfg45(Workload):
    """Convection-zone box shaped like the paper's runs: radial gravity, isentropic shell under a stable layer."""

    @staticmethod
    def g_of_r(r):
        r = np.asarray(r, dtype=np.float64)
        rs = np.maximum(r, 1e-3)
        g = np.where(r < 0.25, -3.0 * (r / 0.25), -3.0 * (0.25 / rs) ** 2)
        tap = np.where(r <= 0.47, 1.0, np.where(r >= 0.49, 0.0, 0.5 * (1.0 + np.cos(math.pi * (r - 0.47) / 0.02))))
        return g * tap

    @classmethod
    def base_table(cls, n=8192, rmax=0.9):
        """(r, g, rho0, p0) fp64 on the table nodes; potential integrated by Simpson (= RK4 for a quadrature)."""
        r = np.linspace(0.0, rmax, n)
        g = cls.g_of_r(r)
        gm = cls.g_of_r(0.5 * (r[1:] + r[:-1]))
        seg = (r[1:] - r[:-1]) / 6.0 * (g[:-1] + 4.0 * gm + g[1:])
        Gc = np.concatenate([[0.0], np.cumsum(seg)])            # int_0^r g
        G = Gc - np.interp(0.25, r, Gc)                          # int_0.25^r g
        G45 = np.interp(0.45, r, G)
        h = 1.5 + G
        rho_shell = (np.maximum(h, 1e-3) / 1.5) ** 1.5
        p_shell = 0.6 * rho_shell ** GAMMA
        h45 = 1.5 + G45
        rho_t = (h45 / 1.5) ** 1.5
        p_t = 0.6 * rho_t ** GAMMA
        a2t = p_t / rho_t
        rho_core = np.exp(G / 0.6)
        rho_top = rho_t * np.exp((G - G45) / a2t)
        rho0 = np.where(r < 0.25, rho_core, np.where(r <= 0.45, rho_shell, rho_top))
        p0 = np.where(r < 0.25, 0.6 * rho_core, np.where(r <= 0.45, p_shell, a2t * rho_top))
        return r, g, rho0, p0

    def _r(self, x, y, z):
        return torch.sqrt((x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2)

    def _hydro(self, x, y, z):
        p = self._p
        r = self._r(x, y, z)
        rho = self._table_interp("rho0", r)
        pr = self._table_interp("p0", r)
        t = torch.clamp((r - 0.27) / 0.16, 0.0, 1.0)
        bump = torch.sin(math.pi * t) ** 2
        u = [_eval_modes(p["vel_modes"][d], (x, y, z), 0.03) * bump for d in range(3)]
        return rho, u[0], u[1], u[2], pr

    def _fv(self, x, y, z):
        wdt = max(1.5 / 512.0, 1.5 * self.dx)
        return 0.5 * (1.0 + torch.tanh((self._r(x, y, z) - 0.45) / wdt))


# ------------------------------------------------------------------------------------------------
def make(cfg: int, n: int | None = None, steps: int | None = None) -> Workload:
    """Workload for BASELINE.json configs[cfg-1]; `n`/`steps` override the size for reduced parity cases."""
    rng = np.random.default_rng(SEED0 + cfg)
    P, R = BC_PERIODIC, BC_REFLECT
    if cfg == 1:
        n = n or 32
        w = _Cfg1(1, "cfg1_periodic_cube", n, steps or 20, 0.8, (P, P, P, P, P, P), None)
        w._p["rho_modes"] = _modes(rng, 3, 2)
        w._p["vel_modes"] = [_modes(rng, 8, 3) for _ in range(3)]
        return w
    if cfg == 2:
        n = n or 128
        dx = 1.0 / n
        nodes = 2 * (n + 2 * NG) + 1
        s0, ds = -NG * dx, 0.5 * dx
        zt = s0 + ds * np.arange(nodes)
        r0, p0 = _Cfg2.base(zt)
        grav = dict(kind=GRAV_CONST_Z, s0=s0, ds=ds, center=(0.0, 0.0, 0.0),
                    g=np.full(nodes, -1.0, dtype=np.float32), rho0=r0.astype(np.float32), p0=p0.astype(np.float32))
        w = _Cfg2(2, "cfg2_stratified_box", n, steps or 100, 0.8, (P, P, P, P, R, R), grav)
        w._p["vel_modes"] = [_modes(rng, 24, 8) for _ in range(3)]
        return w
    if cfg == 3:
        n = n or 256
        w = _Cfg3(3, "cfg3_blast", n, steps or 50, 0.8, (R, R, R, R, R, R), None)
        w._p["if_modes"] = _modes(rng, 8, 4, dims=2)
        return w
    if cfg in (4, 5):
        n = n or (512 if cfg == 4 else 1024)
        # cfg 5 is "the same profiles and seeded perturbations" as cfg 4: same seed
        rng = np.random.default_rng(SEED0 + 4)
        r, g, r0, p0 = _Cfg45.base_table()
        grav = dict(kind=GRAV_RADIAL, s0=0.0, ds=float(r[1] - r[0]), center=(0.5, 0.5, 0.5),
                    g=g.astype(np.float32), rho0=r0.astype(np.float32), p0=p0.astype(np.float32))
        w = _Cfg45(cfg, "cfg%d_convection_zone" % cfg, n, steps or (20 if cfg == 4 else 5), 0.8,
                   (R, R, R, R, R, R), grav)
        w._p["vel_modes"] = [_modes(rng, 32, 8) for _ in range(3)]
        return w
    raise ValueError("cfg must be 1..5")


# ---- NEXT-2: the slotted-disc rotation problem of PAPER.md Fig. 3 / L43 -----------------------------
def slotted_disc(n: int = 100, sub: int = 16, nz: int = 1, revolutions_per_unit_time: float = 1.0):
    """Zalesak's slotted disc in solid-body rotation about the centre of the unit square, as PAPER.md L43 describes it:
    2-D, n x n cells (the paper: 100 x 100), the fractional volume 1 inside the slotted circle and 0 outside, "the
    fractional volumes and higher moments ... computed exactly for a shape with boundaries of zero thickness" — here
    by sub x sub midpoint sub-sampling of the indicator function in every cell (an input recipe, not the method).
    The disc (standard proportions): centre (0.5, 0.75), radius 0.15, slot of width 0.05 cut from below up to y = 0.85.
    Returns fields [15, nz, n, n] float32: rho = 1, p = 1, (u, v) = Omega x (r - centre), w = 0, and the in-plane
    Legendre coefficients of FV (m000, m100, m010, m200, m020, m110; the z ones are zero).  dx = 1/n."""
    dx = 1.0 / n
    om = 2.0 * math.pi * revolutions_per_unit_time
    c = (np.arange(n) + 0.5) * dx
    s = (np.arange(sub) + 0.5) / sub - 0.5                     # sub-cell midpoints in cell units
    xs = (c[:, None] + s[None, :] * dx).reshape(-1)            # n*sub sample coordinates
    X, Y = np.meshgrid(xs, xs, indexing="xy")                  # [y, x]
    inside = ((X - 0.5) ** 2 + (Y - 0.75) ** 2 <= 0.15 ** 2) & ~((np.abs(X - 0.5) <= 0.025) & (Y <= 0.85))
    ind = inside.astype(np.float64).reshape(n, sub, n, sub)    # [cell y, sub y, cell x, sub x]
    P = [np.ones(sub), s, s * s - 1.0 / 12.0]
    f = np.zeros((NF, nz, n, n), dtype=np.float32)
    f[0] = 1.0
    f[4] = 1.0
    f[1] = (-om * (c - 0.5))[None, :, None]                    # u_x = -Omega (y - 1/2)
    f[2] = (om * (c - 0.5))[None, None, :]                     # u_y = +Omega (x - 1/2)
    for k, (a, b, cz) in enumerate(_ABC):
        if cz != 0:
            continue
        mom = np.einsum("jqip,q,p->ji", ind, P[b], P[a]) / (sub * sub) / (_NORM[a] * _NORM[b])
        f[5 + k] = mom[None, :, :]
    return f


def subcell_image(m6, sub: int = 4):
    """The paper's display of Fig. 3: "each grid cell is represented by a 4 x 4 square of subcells in which the
    fractional volume is computed using the 6 low-order moments".  m6: dict or array of the in-plane coefficients
    (m000, m100, m010, m200, m020, m110), each [ny, nx]; returns [ny*sub, nx*sub] sub-cell AVERAGES of the polynomial."""
    m000, m100, m010, m200, m020, m110 = m6
    e = np.arange(sub + 1) / sub - 0.5
    a1 = 0.5 * (e[1:] + e[:-1])                                            # average of P1 over a sub-interval
    a2 = (e[1:] ** 3 - e[:-1] ** 3) / (3.0 * (e[1:] - e[:-1])) - 1.0 / 12.0  # average of P2
    ny, nx = m000.shape
    out = (m000[:, None, :, None] + m100[:, None, :, None] * a1[None, None, None, :] + m010[:, None, :, None] * a1[None, :, None, None]
           + m200[:, None, :, None] * a2[None, None, None, :] + m020[:, None, :, None] * a2[None, :, None, None]
           + m110[:, None, :, None] * a1[None, :, None, None] * a1[None, None, None, :])
    return out.reshape(ny * sub, nx * sub)
