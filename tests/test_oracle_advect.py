"""Pins of the oracle's PPB-only advection mode (Fig. 3: the slotted disc in
solid-body rotation, "linear advection"; reading R22 in DESIGN.md).  The remap itself (P2-P4) is pinned in
test_oracle_pins.py; here: the face mass of the prescribed velocity field, that the hydro state is held fixed, the
link to the full hydro+PPB step, exact translation, conservation, bounds, and the paper's qualitative claims for
Fig. 3 (the disc survives a revolution far better than with a first-order scheme)."""
import numpy as np
import pytest

from oracle import binding as ob
from paper_1810_13416_b200 import workloads as W

P, R = ob.BC_PERIODIC, ob.BC_REFLECT


def _lin_fields(shape, u, grad, c0=0.5, dx=0.1):
    """uniform gas moving with velocity u, FV = c0 + grad . (x - x0) represented exactly (cell mean + first moments)"""
    nz, ny, nx = shape
    f = np.zeros((15,) + shape, dtype=np.float32)
    f[0], f[4] = 1.0, 1.0
    for d in range(3):
        f[1 + d] = u[d]
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    f[5] = c0 + dx * (grad[0] * (x - nx / 2) + grad[1] * (y - ny / 2) + grad[2] * (z - nz / 2))
    for d in range(3):
        f[6 + d] = grad[d] * dx          # m100, m010, m001: slope times the cell width
    return f


def test_pencil_closed_form_uniform_courant_number():
    """uniform u > 0, Courant number sigma: SURVEY 8(c) P4's closed form for the degree-2 family, donor a = cell
    i-1, own b = cell i (worked values: donor == 1, own == 0, sigma = 1/2 -> (1/2, -3/2, 0); sigma = 1/4 ->
    (1/4, -9/8, 45/16))."""
    n, dx = 6, 0.1
    for sigma, exp in ((0.5, (0.5, -1.5, 0.0)), (0.25, (0.25, -9.0 / 8.0, 45.0 / 16.0))):
        u = np.full(n + 8, sigma * dx / 0.01)
        m = np.zeros((10, n + 8))
        m[0, :7] = 1.0                      # cells 0..6 (with ghosts) full, the rest empty: cell 7 receives from a full donor
        out = ob.advect_pencil(0, dx, 0.01, u, m)
        i = 7 - 4                           # interior index of cell 7
        assert np.allclose([out[0][i], out[1][i], out[4][i]], exp, atol=1e-13)


def test_advect_leaves_the_hydro_state_alone_and_conserves_fv():
    rng = np.random.default_rng(2)
    nx, ny, nz = 9, 7, 6
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.0 + rng.random((nz, ny, nx))            # (ignored by the mode: the gas is taken as uniform)
    # a velocity field whose component along each axis does not vary along that axis (like Fig. 3's rotation):
    # every 1-D sweep is then volume preserving, which is what reading R22 assumes
    f[1] = 0.5 * rng.normal(size=(nz, ny, 1))
    f[2] = 0.5 * rng.normal(size=(nz, 1, nx))
    f[3] = 0.5 * rng.normal(size=(1, ny, nx))
    f[4] = 1.0 + rng.random((nz, ny, nx))
    f[5] = 0.3 + 0.4 * rng.random((nz, ny, nx))
    f[6:] = 0.01 * rng.normal(size=(9, nz, ny, nx))
    o = ob.Oracle(nx, ny, nz, 0.1, 1.4, (P,) * 6)
    o.set_state(f)
    s0 = o.get_state()
    for k in range(6):
        o.advect(0.02, k)
    s1 = o.get_state()
    assert np.array_equal(s0[:5], s1[:5])
    assert np.max(np.abs(s1[5] - s0[5])) > 1e-3                       # ... but FV moved
    assert abs(s1[5].sum() - s0[5].sum()) < 1e-12 * s0[5].size        # sum of cell means (rho = 1): conserved
    assert s1[5].min() >= 0.0 and s1[5].max() <= 1.0


def test_full_step_and_advect_mode_agree_on_a_uniform_flow():
    """uniform rho, u, p on a periodic box: the hydro step preserves the state and its mass fluxes are rho*u, so the
    FV update of the full PPM+PPB step must equal the PPB-only mode's (the mass coordinate cancels rho)."""
    rng = np.random.default_rng(3)
    nx, ny, nz = 8, 8, 8
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0], f[4] = 1.75, 0.9
    f[1], f[2], f[3] = 0.4, -0.3, 0.2
    f[5] = 0.3 + 0.4 * rng.random((nz, ny, nx))
    f[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    res = []
    for mode in ("step", "advect"):
        o = ob.Oracle(nx, ny, nz, 0.1, 1.4, (P,) * 6)
        o.set_state(f)
        for k in (0, 5, 3):
            getattr(o, mode)(0.03, k)
        res.append(o.get_state())
    assert np.max(np.abs(res[0][5:] - res[1][5:])) < 1e-12
    assert np.max(np.abs(res[0][:5] - res[1][:5])) < 1e-13


def test_linear_field_translates_exactly():
    nx, ny, nz, dx = 16, 14, 13, 0.125                  # dyadic numbers: the fp32 input is exact
    u, grad = (0.7, -0.4, 0.3), (0.125, -0.125, 0.0625)
    f = _lin_fields((nz, ny, nx), u, grad, dx=dx)
    o = ob.Oracle(nx, ny, nz, dx, 1.4, (P,) * 6)
    o.set_state(f)
    dt, steps = 0.04, 3
    for k in range(steps):
        o.advect(dt, 2 * k)
    s = o.get_state()
    shift = sum(-grad[d] * u[d] * dt * steps for d in range(3))
    inner = (slice(4, nz - 4), slice(4, ny - 4), slice(4, nx - 4))    # away from the periodic seam of the linear ramp
    assert np.max(np.abs(s[5][inner] - (f[5].astype(np.float64)[inner] + shift))) < 1e-13
    for d in range(3):
        assert np.max(np.abs(s[6 + d][inner] - grad[d] * dx)) < 1e-13
    assert np.max(np.abs(s[9:][(slice(None),) + inner])) < 1e-12


def _l1(a, b):
    return np.abs(a - b).sum() / a.size


def test_slotted_disc_one_revolution_fig3():
    """PAPER.md Fig. 3 / L43 on the paper's grid (100 x 100, 6 moments): after one revolution the disc is back in
    place.  No numbers are printed in the paper, so the pins are relative: the PPB result is several times
    closer to the initial state than first-order (donor-cell: moments dropped every step) advection of the same
    field, the slot is still open and the bridge still full, FV stays in [0,1] and its integral is conserved."""
    n = 100
    f = W.slotted_disc(n)
    steps = 1256                                   # CFL = Omega*0.5*sqrt(2)*dt/dx ~ 0.35 at the corner
    dt = 1.0 / steps
    res = {}
    for scheme in ("ppb", "donor"):
        # periodic faces: u_x does not depend on x (nor u_y on y), so the wrap is seamless along every sweep and each
        # sweep is volume preserving (a mirror wall would squeeze the uniform gas of reading R22 in the wall cells)
        o = ob.Oracle(n, n, 1, 1.0 / n, 1.4, (P,) * 6)
        o.set_state(f)
        for k in range(steps):
            o.advect(dt, 0 if k % 2 == 0 else 2)   # xyz / yxz alternating (z does nothing: u_z = 0)
            if scheme == "donor":
                for q in range(6, 15):
                    o.raw_field(q)[:] = 0.0
        res[scheme] = o.get_state()
    m0 = f[5, 0].astype(np.float64)
    ppb, donor = res["ppb"][5, 0], res["donor"][5, 0]
    assert abs(ppb.sum() - m0.sum()) < 1e-10 * n * n
    assert ppb.min() >= 0.0 and ppb.max() <= 1.0
    e_ppb, e_donor = _l1(ppb, m0), _l1(donor, m0)
    assert e_ppb < 0.2 * e_donor and e_ppb < 0.012, (e_ppb, e_donor)       # measured: 0.0103 vs 0.0658
    # the slot (x = 0.5, y in 0.62..0.80) is still empty and the solid part beside it (x = 0.44 / 0.56) still full
    ys = slice(64, 78)
    assert ppb[ys, 49:51].max() < 0.12 and donor[ys, 49:51].max() > 0.3
    assert ppb[ys, 43:45].min() > 0.9 and ppb[ys, 55:57].min() > 0.9
    # sub-cell picture of the paper (4 x 4 per cell): same integral as the cell means
    s = res["ppb"]
    img = W.subcell_image([s[5, 0], s[6, 0], s[7, 0], s[9, 0], s[10, 0], s[12, 0]])
    assert img.shape == (400, 400) and abs(img.mean() - ppb.mean()) < 1e-12
