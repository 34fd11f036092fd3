"""Pins of the oracle's fully 3-D shock-flattening mode ("a fully 3-D treatment
of the shock dissipation"; reading R5b in DESIGN.md).  The 1-D detector oracle_h4_ftilde is pinned in
test_oracle_pins.py; here the pins are on what the 3-D mode adds: the max over the three directions, the boundary
images, which sweep sees which coefficient, and the cases where the mode must reduce to the 1-D one."""
import numpy as np
import pytest

from oracle import binding as ob
from paper_1810_13416_b200 import workloads as W

from test_oracle_invariants import _permute_fields

P, R = ob.BC_PERIODIC, ob.BC_REFLECT
G = 1.4


def _shock_fields(shape, axis, rng=None, amp=0.0):
    """a Mach ~3 two-cell shock profile moving along `axis` (0=x), uniform across it; optional transverse noise"""
    nz, ny, nx = shape
    n = (nx, ny, nz)[axis]
    s = np.arange(n)
    # post-shock | pre-shock (gamma = 1.4, Mach 3 into gas at rest): rho 3.857 / 1, u 2.629 / 0, p 10.33 / 1
    w = 0.5 * (1 - np.tanh((s - n / 2 + 0.5) / 0.6))
    prof = lambda a, b: b + (a - b) * w
    sh = [1, 1, 1]
    sh[2 - axis] = n
    f = np.zeros((15,) + shape, dtype=np.float32)
    f[0] = prof(3.857, 1.0).reshape(sh)
    f[1 + axis] = prof(2.629, 0.0).reshape(sh)
    f[4] = prof(10.33, 1.0).reshape(sh)
    f[5] = 0.5
    if rng is not None:
        f[0] *= 1.0 + amp * rng.random(shape)
        f[4] *= 1.0 + amp * rng.random(shape)
    return f


def _brute_force_F(f, bc, gamma):
    """F~ from the definition, with numpy index arithmetic written independently of the oracle's image_cell"""
    rho, p = f[0].astype(np.float64), f[4].astype(np.float64)
    nz, ny, nx = rho.shape
    ext = (nx, ny, nz)
    F = np.zeros_like(rho)
    c = np.sqrt(gamma * p / rho)
    for d in range(3):
        ax = 2 - d
        n = ext[d]
        u = f[1 + d].astype(np.float64)

        def take(a, o, odd=False):
            idx = np.arange(n) + o
            sg = np.ones(n)
            if bc[2 * d] == P:
                idx = idx % n
            else:
                lo, hi = idx < 0, idx >= n
                sg[lo | hi] = -1.0
                idx = np.where(lo, -1 - idx, np.where(hi, 2 * n - 1 - idx, idx))
            out = np.take(a, idx, axis=ax)
            if odd:
                shp = [1, 1, 1]
                shp[ax] = n
                out = out * sg.reshape(shp)
            return out

        p5 = [take(p, o) for o in (-2, -1, 0, 1, 2)]
        um, up = take(u, -1, True), take(u, 1, True)
        for idx in np.ndindex(rho.shape):
            F[idx] = max(F[idx], ob.h4_ftilde([a[idx] for a in p5], um[idx], up[idx], c[idx]))
    return F


@pytest.mark.parametrize("bc", [(P,) * 6, (R,) * 6, (P, P, R, R, P, P)])
def test_detector_field_is_the_max_over_the_three_directions(bc):
    rng = np.random.default_rng(5)
    nx, ny, nz = 7, 6, 5
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.0 + rng.random((nz, ny, nx))
    f[1:4] = 1.5 * rng.normal(size=(3, nz, ny, nx))       # strongly convergent in places
    f[4] = np.exp(2.5 * rng.normal(size=(nz, ny, nx)))      # pressure jumps of every size
    f[5] = 0.5
    o = ob.Oracle(nx, ny, nz, 0.1, G, bc)
    o.set_state(f)
    o.set_flatten3d(True)
    F = o.flatten3d_field()
    ref = _brute_force_F(f, bc, G)
    assert 0.05 < (ref > 0).mean() < 0.95 and ref.max() == 1.0          # the case exercises on, off and ramps
    assert np.max(np.abs(F - ref)) < 1e-14


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_flow_varying_along_one_axis_reduces_to_the_1d_mode(axis):
    """a planar shock along `axis`, uniform across it: the other two detectors vanish, and the sweeps across the
    shock see flat data, so F~ = f~ of that axis and the step equals the 1-D mode's (first sweep along the shock)."""
    shape = [4, 4, 4]
    shape[2 - axis] = 24
    f = _shock_fields(tuple(shape), axis)
    bc = [P] * 6
    bc[2 * axis] = bc[2 * axis + 1] = R
    order = {0: 0, 1: 2, 2: 4}[axis]         # xyz, yxz, zxy: the shock direction first
    res = []
    for mode in (False, True):
        o = ob.Oracle(shape[2], shape[1], shape[0], 1.0 / 24, G, bc)
        o.set_state(f)
        o.set_flatten3d(mode)
        if mode:
            F = o.flatten3d_field()
            assert F.max() > 0.8 and (F > 0.5).sum() >= 16            # flattening is really on in the shock
        for s in range(4):
            o.step(0.25 * o.cfl_dt(0.8), order)
        res.append(o.get_state())
    assert np.max(np.abs(res[0] - res[1])) < 1e-13


def test_smooth_flow_is_untouched_by_the_3d_mode():
    w = W.make(1, n=16)
    res = []
    for mode in (False, True):
        o = ob.Oracle(16, 16, 16, w.dx, w.gamma, w.bc, None)
        o.set_state(w.fields().numpy())
        o.set_flatten3d(mode)
        if mode:
            assert not o.flatten3d_field().any()
        for s in range(3):
            o.step(o.cfl_dt(0.8), 5 * (s % 2))
        res.append(o.get_state())
    assert np.array_equal(res[0], res[1])


def test_transverse_sweeps_see_the_shock_only_in_the_3d_mode():
    """x shock with transverse (y, z) noise: in the 1-D mode the y sweep does not know about the shock and keeps its
    parabolas; in the 3-D mode the coefficient of the x detector flattens them.  Checked on one pencil through the
    public 1-D routine: with ft_ext = 1 inside the shock the pencil update is the first-order (donor-cell) one,
    i.e. it equals the update of the same pencil with every parabola forced flat."""
    rng = np.random.default_rng(9)
    n = 12
    q5 = np.zeros((5, n + 8))
    q5[0] = 1.0 + 0.2 * rng.random(n + 8)
    q5[1] = 0.1 * rng.normal(size=n + 8)
    q5[2:4] = 0.1 * rng.normal(size=(2, n + 8))
    q5[4] = 1.0 + 0.2 * rng.random(n + 8)
    m10 = np.zeros((10, n + 8))
    m10[0] = 0.5
    a, _ = ob.sweep_pencil(1, 0.1, 0.02, G, q5, m10)
    b, _ = ob.sweep_pencil(1, 0.1, 0.02, G, q5, m10, ft_ext=np.zeros(n + 8))
    c, _ = ob.sweep_pencil(1, 0.1, 0.02, G, q5, m10, ft_ext=np.ones(n + 8))
    assert np.array_equal(a, b)                      # smooth-ish data: the 1-D detector is off, like ft_ext = 0
    assert np.max(np.abs(a - c)) > 1e-5              # fully flattened parabolas give a different (first-order) update
    # donor-cell check of c for the density: with flat parabolas the traced states are the cell means, so the
    # face states of the Riemann problem are (cell j-1, cell j); redo that with the public Riemann routine
    flux = np.zeros(n + 9)
    for fidx in range(4, n + 5):
        L = [q5[0][fidx - 1], q5[1][fidx - 1], q5[2][fidx - 1], q5[3][fidx - 1], q5[4][fidx - 1]]
        Rr = [q5[0][fidx], q5[1][fidx], q5[2][fidx], q5[3][fidx], q5[4][fidx]]
        s, _, _ = ob.h7_riemann(L, Rr, G)
        flux[fidx] = s[0] * s[1]
    rho_new = q5[0][4:n + 4] - 0.02 / 0.1 * (flux[5:n + 5] - flux[4:n + 4])
    assert np.max(np.abs(c[0] - rho_new)) < 1e-13


def test_3d_mode_axis_permutation_symmetry():
    rng = np.random.default_rng(4)
    nx, ny, nz = 10, 8, 6
    f = _shock_fields((nz, ny, nx), 0, rng, 0.3)
    f[2:4] = 0.5 * rng.normal(size=(2, nz, ny, nx))
    orders = [(0, 1, 2), (0, 2, 1), (1, 0, 2), (1, 2, 0), (2, 0, 1), (2, 1, 0)]
    o = ob.Oracle(nx, ny, nz, 0.1, G, (P,) * 6)
    o.set_state(f)
    o.set_flatten3d(True)
    assert o.flatten3d_field().max() > 0.5
    o.step(0.004, 0)
    ref = o.get_state()
    for perm in ((1, 2, 0), (2, 0, 1), (1, 0, 2)):
        fp = np.ascontiguousarray(_permute_fields(f, perm))
        nzp, nyp, nxp = fp.shape[1:]
        o2 = ob.Oracle(nxp, nyp, nzp, 0.1, G, (P,) * 6)
        o2.set_state(fp)
        o2.set_flatten3d(True)
        inv = [perm.index(d) for d in range(3)]
        o2.step(0.004, orders.index(tuple(inv)))
        assert np.max(np.abs(o2.get_state() - _permute_fields(ref, perm))) < 1e-12


def test_3d_mode_keeps_conservation_and_uniform_state():
    rng = np.random.default_rng(6)
    n = 12
    f = _shock_fields((n, n, n), 0, rng, 0.2)
    f[2:4] = 0.3 * rng.normal(size=(2, n, n, n))
    o = ob.Oracle(n, n, n, 1.0 / n, G, (P,) * 6)
    o.set_state(f)
    o.set_flatten3d(True)
    c0 = o.reduce_conserved()
    for s in range(4):
        o.step(0.5 * o.cfl_dt(0.8), s)
    c1 = o.reduce_conserved()
    assert np.max(np.abs(c1 - c0) / np.maximum(np.abs(c0), 1e-3)) < 1e-12
    u = np.zeros((15, 5, 6, 7), dtype=np.float32)
    u[0], u[4], u[5] = 1.3, 0.7, 0.25
    o = ob.Oracle(7, 6, 5, 0.1, G, (R,) * 6)
    o.set_state(u)
    o.set_flatten3d(True)
    o.step(0.01, 3)
    g = o.get_state()
    assert np.array_equal(g[:4], u[:4].astype(np.float64)) and np.array_equal(g[5], u[5].astype(np.float64))
