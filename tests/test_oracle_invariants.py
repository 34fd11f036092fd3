"""Invariants the oracle must satisfy (BASELINE.json north_star; SURVEY.md 8(c) C9 rows "H0-H9 together",
"P1-P4 in 3-D", "C6, C7"): uniform/hydrostatic preservation, conservation, convergence to the exact
Riemann solution, smooth-flow convergence order, exact translation of a linear FV field, axis-permutation
symmetry, FV in [0,1], window == full grid."""
import math

import numpy as np
import pytest

from oracle import binding as ob
from paper_1810_13416_b200 import workloads as W

import exact_riemann as ex

P, R, O = ob.BC_PERIODIC, ob.BC_REFLECT, ob.BC_OPEN
G = 5.0 / 3.0


def _mk(nx, ny, nz, bc, dx=None, gamma=G, grav=None, org=(0, 0, 0)):
    return ob.Oracle(nx, ny, nz, dx if dx is not None else 1.0 / nx, gamma, bc, grav, org=org)


def _fields(shape, rho=1.0, u=(0, 0, 0), p=1.0, m=None):
    f = np.zeros((15,) + shape, dtype=np.float32)
    f[0], f[1], f[2], f[3], f[4] = rho, u[0], u[1], u[2], p
    if m is not None:
        for k in range(10):
            f[5 + k] = m[k]
    return f


# ---------------------------------------------------------------- preservation ---------------------
@pytest.mark.parametrize("bc", [(P,) * 6, (R,) * 6, (P, P, R, R, P, P)])
def test_uniform_state_preserved_bitwise(bc):
    o = _mk(8, 6, 5, bc)
    f = _fields((5, 6, 8), rho=1.7, u=(0.3, -0.2, 0.1) if bc == (P,) * 6 else (0, 0, 0), p=0.9,
                m=[0.4, 0, 0, 0, 0, 0, 0, 0, 0, 0])
    o.set_state(f)
    for s in range(3):
        o.step(0.02, s)
    g = o.get_state()
    f64 = f.astype(np.float64)
    if bc == (P,) * 6:      # moving uniform state: conservative update -> preserved to round-off
        assert np.max(np.abs(g - f64)) < 2e-14
    else:                   # at rest: rho, u, FV bit for bit; p goes through E = p/(gamma-1) -> 1 ulp
        assert np.array_equal(g[:4], f64[:4]) and np.array_equal(g[5], f64[5])
        # (the P2-projection of a constant is 180 x quadrature round-off)
        assert np.max(np.abs(g[4] - f64[4])) <= 4e-16 and np.max(np.abs(g[6:])) < 1e-14


def test_hydrostatic_base_state_preserved_bitwise_const_z_and_radial():
    for cfg, n in ((2, 16), (4, 20)):
        w = W.make(cfg, n=n)
        o = ob.Oracle(n, n, n, w.dx, w.gamma, w.bc, w.grav)
        f = w.fields().numpy()
        f[1:4] = 0.0
        o.set_state(f)
        for k in (0, 4):
            o.raw_field(k)[:] = 0.0          # exactly zero perturbation
        ref = o.get_state()
        assert ref[0].max() / ref[0].min() > 1.3         # the base state really is stratified
        dt = o.cfl_dt(0.8)
        # well-balanced: every face has u^ = 0 and p^' = 0, so after a sweep rho' and the velocities are
        # EXACTLY zero; p is rebuilt from E = p/(gamma-1), i.e. it is preserved to the last bit
        o.sweep(2, dt)
        for k in range(4):
            assert not o.raw_field(k).any()
        assert np.max(np.abs(o.raw_field(4))) <= 2.3e-16
        for s in range(3):
            o.step(dt, s)
        for k in range(5):
            assert np.max(np.abs(o.raw_field(k))) <= 5e-15      # only that last-bit noise evolves


# ---------------------------------------------------------------- conservation ---------------------
def test_conservation_periodic_config1():
    w = W.make(1)
    o = ob.Oracle(w.n, w.n, w.n, w.dx, w.gamma, w.bc, None)
    o.set_state(w.fields().numpy())
    c0 = o.reduce_conserved()
    raw = o.get_state()
    scale_mom = np.sum(np.abs(raw[0] * raw[1])) * w.dx ** 3
    for s in range(6):
        o.step(o.cfl_dt(0.8), 0 if s % 2 == 0 else 5)
    c1 = o.reduce_conserved()
    assert abs(c1[0] - c0[0]) <= 1e-13 * c0[0]
    assert abs(c1[4] - c0[4]) <= 1e-13 * c0[4]
    assert abs(c1[5] - c0[5]) <= 1e-13 * c0[5]
    assert np.all(np.abs(c1[1:4] - c0[1:4]) <= 1e-13 * scale_mom)
    fv = o.get_state()[5]
    assert fv.min() >= 0.0 and fv.max() <= 1.0


def test_closed_box_with_reflecting_walls_conserves_mass():
    w = W.make(3, n=16)
    o = ob.Oracle(16, 16, 16, w.dx, w.gamma, w.bc, None)
    o.set_state(w.fields().numpy())
    c0 = o.reduce_conserved()
    for s in range(4):
        o.step(o.cfl_dt(0.8), s)
    c1 = o.reduce_conserved()
    assert abs(c1[0] - c0[0]) <= 1e-12 * c0[0]
    assert abs(c1[5] - c0[5]) <= 1e-12 * c0[5]
    assert abs(c1[4] - c0[4]) <= 1e-12 * c0[4]     # g = 0: walls do no work


def test_cfl_and_conserved_hand_values_on_2x2x2():
    o = _mk(2, 2, 2, (P,) * 6, dx=0.5, gamma=1.4)
    f = _fields((2, 2, 2), rho=2.0, u=(0.5, -1.5, 0.25), p=1.4 * 2.0 / 1.4)   # c = sqrt(1.4*2/2) = sqrt(1.4)
    f[0, 1, 1, 1] = 8.0                                                          # one heavy cell: c = sqrt(1.4*2/8)
    f[5] = 0.25
    o.set_state(f)
    assert o.cfl_dt(0.8) == pytest.approx(0.8 * 0.5 / (1.5 + math.sqrt(1.4)), rel=1e-14)
    c = o.reduce_conserved()
    dv = 0.125
    mass = (7 * 2.0 + 8.0) * dv
    assert c[0] == pytest.approx(mass, rel=1e-14)
    assert c[1:4] == pytest.approx([mass * 0.5, mass * -1.5, mass * 0.25], rel=1e-14)
    assert c[4] == pytest.approx(8 * dv * 2.0 / 0.4 + 0.5 * mass * (0.25 + 2.25 + 0.0625), rel=1e-14)
    assert c[5] == pytest.approx(0.25 * mass, rel=1e-14)


# ---------------------------------------------------------------- 1-D convergence ------------------
def _run_1d(n, rho, u, p, gamma, t_end, cfl, bc):
    o = _mk(n, 1, 1, bc + (P, P, P, P), dx=1.0 / n, gamma=gamma)
    f = _fields((1, 1, n), rho=1.0)
    f[0, 0, 0], f[1, 0, 0], f[4, 0, 0] = rho, u, p
    o.set_state(f)
    t = 0.0
    while t < t_end - 1e-14:
        dt = min(o.cfl_dt(cfl), t_end - t)
        o.sweep(0, dt)
        t += dt
    return o.get_state()[:, 0, 0, :]


def test_sod_shock_tube_converges_to_exact_solution_first_order():
    g = 1.4
    errs = []
    for n in (100, 200, 400):
        x = (np.arange(n) + 0.5) / n
        left = x < 0.5
        s = _run_1d(n, np.where(left, 1.0, 0.125), np.zeros(n), np.where(left, 1.0, 0.1), g, 0.2, 0.8, (R, R))
        exact = ex.profile(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g, x, 0.5, 0.2)
        errs.append(np.mean(np.abs(s[0] - exact[:, 0])))
        assert np.mean(np.abs(s[1] - exact[:, 1])) < 6.0 / n
        assert np.mean(np.abs(s[4] - exact[:, 2])) < 3.0 / n
    assert errs[0] < 0.012
    assert errs[1] < errs[0] / 1.6 and errs[2] < errs[1] / 1.6      # ~ first order in L1


def test_smooth_entropy_wave_convergence_order():
    # rho = 1 + 0.2 sin(2 pi x), u = 1, p = 1 translates unchanged.  PAPER.md L27/L33: with the limiter
    # inactive in smooth flow the scheme keeps its formal accuracy, also as the Courant number -> 0.
    def err(n, cfl):
        x = (np.arange(n) + 0.5) / n
        h = 0.5 / n
        avg = lambda x0: 1.0 + 0.2 * (np.cos(2 * np.pi * (x0 - h)) - np.cos(2 * np.pi * (x0 + h))) / (2 * np.pi * 2 * h)
        s = _run_1d(n, avg(x), np.ones(n), np.ones(n), G, 0.5, cfl, (P, P))
        return np.mean(np.abs(s[0] - avg(x - 0.5)))
    e = [err(n, 0.8) for n in (16, 32, 64)]
    assert math.log2(e[0] / e[1]) > 2.5 and math.log2(e[1] / e[2]) > 2.5
    e2 = [err(n, 0.1) for n in (16, 32)]
    assert math.log2(e2[0] / e2[1]) > 2.5
    assert e2[1] < 4 * e[1]          # accuracy does not collapse as the Courant number shrinks (L33)


# ---------------------------------------------------------------- PPB in 3-D -----------------------
def test_linear_fv_field_translates_exactly_under_uniform_velocity():
    n = 12
    dx = 1.0 / n
    o = _mk(n, n, n, (P,) * 6)
    vel = (0.31, -0.22, 0.17)
    a, gx, gy, gz = 0.5, 0.25, -0.15, 0.2
    x = (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    m = np.zeros((10, n, n, n))
    m[0] = a + gx * (X - 0.5) + gy * (Y - 0.5) + gz * (Z - 0.5)
    m[1], m[2], m[3] = gx * dx, gy * dx, gz * dx
    f = _fields((n, n, n), rho=1.3, u=vel, p=0.8, m=m)
    o.set_state(f)
    f32 = f.astype(np.float64)
    dt, t = 0.7 * dx, 0.0
    for s in range(2):
        o.step(dt, s * 5)
        t += dt
    g = o.get_state()
    exp0 = f32[5] - (gx * vel[0] + gy * vel[1] + gz * vel[2]) * t
    sl = (slice(5, n - 5),) * 3             # away from the periodic seam (the linear field jumps there)
    assert np.max(np.abs(g[5][sl] - exp0[sl])) < 1e-7      # fp32 input rounding only
    for k, v in ((6, gx * dx), (7, gy * dx), (8, gz * dx)):
        assert np.max(np.abs(g[k][sl] - np.float32(v))) < 1e-7
    for k in range(9, 15):
        assert np.max(np.abs(g[k][sl])) < 1e-7
    assert np.array_equal(g[0], f32[0]) or np.max(np.abs(g[0] - 1.3)) < 1e-6


def test_uniform_fv_stays_uniform_in_compressible_flow():
    w = W.make(3, n=16)
    o = ob.Oracle(16, 16, 16, w.dx, w.gamma, w.bc, None)
    f = w.fields().numpy()
    f[5:] = 0.0
    f[5] = 0.37
    o.set_state(f)
    for s in range(3):
        o.step(o.cfl_dt(0.8), s)
    g = o.get_state()
    assert g[0].max() / g[0].min() > 100 and np.abs(g[1:4]).max() > 1.0     # the flow is violent
    assert np.max(np.abs(g[5] - np.float32(0.37))) < 1e-13
    assert np.max(np.abs(g[6:])) < 1e-13


def test_fv_stays_in_unit_interval_sharp_interface():
    n = 16
    w = W.make(1, n=n)
    o = ob.Oracle(n, n, n, w.dx, w.gamma, w.bc, None)
    f = w.fields().numpy()
    # sharp slab: cell means exactly 0 / 1, higher coefficients zero -> exercises the P2 scaling
    f[5:] = 0.0
    f[5, 4:9] = 1.0
    f[1:4] *= 10.0
    o.set_state(f)
    for s in range(8):
        o.step(o.cfl_dt(0.8), s % 6)
    fv = o.get_state()[5]
    assert fv.min() >= 0.0 and fv.max() <= 1.0
    assert fv.max() > 0.99 and fv.min() < 0.01


# ---------------------------------------------------------------- symmetry -------------------------
_PERM_M = {  # coefficient permutation when axes are relabelled x->y->z->x, i.e. new(y) = old(x) ...
}


def _permute_fields(f, perm):
    """relabel axes: new axis a = old axis perm[a] (axes numbered x=0,y=1,z=2).  f: [15, nz, ny, nx]."""
    abc = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (0, 2, 0), (0, 0, 2), (1, 1, 0), (1, 0, 1), (0, 1, 1)]
    # array axes order is (z, y, x) = (2, 1, 0): array axis index for physical axis a is 2 - a
    tr = [2 - perm[2 - ax] for ax in range(3)]
    out = np.empty((15,) + tuple(f.shape[1 + t] for t in tr), dtype=f.dtype)
    T = lambda a: np.transpose(a, tr)
    out[0], out[4] = T(f[0]), T(f[4])
    for a in range(3):
        out[1 + a] = T(f[1 + perm[a]])
    for k, e in enumerate(abc):
        # new exponent along new axis a = old exponent along old axis perm[a]
        for k2, e2 in enumerate(abc):
            if all(e[a] == e2[perm[a]] for a in range(3)):
                out[5 + k] = T(f[5 + k2])
    return out


def test_axis_permutation_symmetry():
    rng = np.random.default_rng(3)
    nx, ny, nz = 10, 8, 6
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    f[0] = 1.0 + 0.3 * rng.random((nz, ny, nx))
    f[1:4] = 0.3 * rng.normal(size=(3, nz, ny, nx))
    f[4] = 0.8 + 0.3 * rng.random((nz, ny, nx))
    f[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    f[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    orders = [(0, 1, 2), (0, 2, 1), (1, 0, 2), (1, 2, 0), (2, 0, 1), (2, 1, 0)]
    o = ob.Oracle(nx, ny, nz, 0.1, G, (P,) * 6)
    o.set_state(f)
    o.step(0.03, 0)           # xyz
    ref = o.get_state()
    for perm in ((1, 2, 0), (2, 0, 1), (1, 0, 2)):
        fp = np.ascontiguousarray(_permute_fields(f, perm))
        nzp, nyp, nxp = fp.shape[1:]
        o2 = ob.Oracle(nxp, nyp, nzp, 0.1, G, (P,) * 6)
        o2.set_state(fp)
        # old sweep order x,y,z: old axis d is new axis a with perm[a] == d
        inv = [perm.index(d) for d in range(3)]
        o2.step(0.03, orders.index(tuple(inv)))
        got = o2.get_state()
        exp = _permute_fields(ref, perm)
        assert np.max(np.abs(got - exp)) < 1e-13


def test_mirror_symmetry_reflecting_box():
    rng = np.random.default_rng(5)
    n = 8
    f = np.zeros((15, n, n, n), dtype=np.float32)
    f[0] = 1.0 + 0.3 * rng.random((n, n, n))
    f[1:4] = 0.3 * rng.normal(size=(3, n, n, n))
    f[4] = 0.8 + 0.3 * rng.random((n, n, n))
    f[5] = 0.5
    f[6] = 0.01 * rng.normal(size=(n, n, n))
    o = ob.Oracle(n, n, n, 0.1, G, (R,) * 6)
    o.set_state(f)
    o.step(0.03, 0)
    ref = o.get_state()
    fm = f[:, :, :, ::-1].copy()
    fm[1] *= -1
    for k in (6, 12, 13):      # m100, m110, m101 odd in x
        fm[k] *= -1
    o2 = ob.Oracle(n, n, n, 0.1, G, (R,) * 6)
    o2.set_state(fm)
    o2.step(0.03, 0)
    got = o2.get_state()[:, :, :, ::-1].copy()
    got[1] *= -1
    for k in (6, 12, 13):
        got[k] *= -1
    assert np.max(np.abs(got - ref)) < 1e-13


# ---------------------------------------------------------------- window mode ----------------------
def test_window_reproduces_full_grid():
    w = W.make(4, n=32)
    n = 32
    full = ob.Oracle(n, n, n, w.dx, w.gamma, w.bc, w.grav)
    f = w.fields().numpy()
    full.set_state(f)
    steps, dt = 2, None
    dt = full.cfl_dt(0.8)
    lo, hi = (0, 6, 10), (20, 26, 32)          # touches the xlo wall and the zhi wall
    bc = (R, O, O, O, O, R)
    win = ob.Oracle(hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2], w.dx, w.gamma, bc, w.grav, org=lo)
    fw = w.fields(lo, hi).numpy()
    assert np.array_equal(fw, f[:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]])     # generator is window-exact
    win.set_state(fw)
    for s in range(steps):
        full.step(dt, s * 5)
        win.step(dt, s * 5)
    a = NG = 4 * steps
    gf = full.get_state()[:, lo[2] + a:hi[2], lo[1] + a:hi[1] - a, lo[0]:hi[0] - a]
    gw = win.get_state()[:, a:, a:-a, :-a]
    assert np.array_equal(gf, gw)


# ---------------------------------------------------------------- parity floor of an fp32 state ----
def test_fp32_state_storage_sets_the_parity_floor():
    """Evidence for DESIGN.md reading R20a.  Run the fp64 oracle twice on config 1, once rounding the STATE to
    fp32 after every sweep (the state is fp32) and nothing else.  The hydro variables and FV
    (scaled by max |m000|) stay ~1e-6 apart, but a coefficient that is ~0 by symmetry moves by >1e-5 of its
    own maximum — so 'relative to the field's own maximum' is not a usable norm for the ten coefficients."""
    from parity_norms import max_rel
    w = W.make(1)
    f = w.fields().numpy()
    A = ob.Oracle(w.n, w.n, w.n, w.dx, w.gamma, w.bc, None)
    B = ob.Oracle(w.n, w.n, w.n, w.dx, w.gamma, w.bc, None)
    A.set_state(f)
    B.set_state(f)
    orders = [(0, 1, 2), (2, 1, 0)]
    for s in range(5):
        dt = A.cfl_dt(0.8)
        A.step(dt, 0 if s % 2 == 0 else 5)
        for d in orders[s % 2]:
            B.sweep(d, dt)
            for k in range(15):
                r = B.raw_field(k)
                r[:] = r.astype(np.float32).astype(np.float64)
    a, b = A.get_state(), B.get_state()
    e = max_rel(b, a)
    assert max(e.values()) < 5e-6
    own = max(np.abs(b[k] - a[k]).max() / np.abs(a[k]).max() for k in range(6, 15))
    assert own > 1e-5
