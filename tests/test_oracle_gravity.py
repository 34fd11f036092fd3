"""Pins of the oracle's gravity / base-state source terms (SURVEY.md 8(c) C1, H6 half-step sources, H9 time-centred
sources; "advance ... perturbations to this initial state ... explicitly cancel out all large
contributions ... valid for perturbations of any size").

The hydrostatic-preservation test (tests/test_oracle_invariants.py) has u = 0 and rho' = p' = 0, where every one of
these terms multiplies zero.  Each test here is a closed form or an invariant that the MATHEMATICS fixes and that a
plausible one-line mistake breaks (the mutations that were tried are listed in DESIGN.md section 7):

  (a) free fall: uniform gas in a uniform field, no base state      -> u(t) = u(0) + g t exactly, rho, p, FV unchanged
      the same with a NON-uniform density (an entropy wave)         -> u stays uniform, exactly
                                                                       (H9 momentum + energy sources, their time centring)
      harmonic RADIAL field, one tiny step from rest                -> du = dt g(r) (X - centre)/r   (base_at direction)
  (b) split invariance: the same physical state carried with table (rho0, p0, g) and with (rho0/2, p0/2, g) — both
      hydrostatic — agree to truncation order under refinement      (H6 tracing sources -u d(rho0,p0)/dx, g rho'/rho)
  (c) energy budget: closed box, fixed g(z): sum (E + rho Phi) constant to second order, mass exact
  (d) mirror sign of g: a reflecting-wall run equals the doubled periodic run of the even-extended state
  (e) table_lookup off the nodes: a table linear in s is reproduced exactly (and extrapolated linearly past its end)
"""
import math

import numpy as np
import pytest

from oracle import binding as ob

P, R, O = ob.BC_PERIODIC, ob.BC_REFLECT, ob.BC_OPEN
G = 5.0 / 3.0
NG = 4


def _const_z_table(nz, dx, g_of_z, rho0_of_z, p0_of_z, z_of_node=None):
    """CONST_Z table: a node on every cell centre and face, the 4 ghost cells included (include/ppm.h)"""
    n = 2 * (nz + 2 * NG) + 1
    s0, ds = -NG * dx, 0.5 * dx
    z = s0 + ds * np.arange(n)
    if z_of_node is not None:
        z = z_of_node(z)
    return dict(kind=ob.GRAV_CONST_Z, s0=s0, ds=ds, center=(0.0, 0.0, 0.0),
                g=np.asarray(g_of_z(z) + 0 * z, dtype=np.float32), rho0=np.asarray(rho0_of_z(z) + 0 * z, dtype=np.float32),
                p0=np.asarray(p0_of_z(z) + 0 * z, dtype=np.float32))


def _fields(shape, rho=1.0, u=(0.0, 0.0, 0.0), p=1.0, fv=0.5):
    f = np.zeros((15,) + shape, dtype=np.float32)
    f[0], f[1], f[2], f[3], f[4], f[5] = rho, u[0], u[1], u[2], p, fv
    return f


# ---------------------------------------------------------------- (a) free fall ---------------------------------------
@pytest.mark.parametrize("u0", [(0.0, 0.0, 0.0), (0.2, -0.1, 0.15)])
def test_free_fall_in_a_uniform_field_is_exact(u0):
    """Uniform gas, CONST_Z table with constant g and rho0 = p0 = 0 (so rho' = rho), periodic box.  Every flux is
    uniform, so only the sources act: u_z = u_z(0) + g t to round-off after any number of steps, rho, p, FV unchanged,
    and the total energy changes by exactly the change of kinetic energy (H9: time-centred momentum source
    dt (rho'^n + rho'^n+1)/2 g and energy source dt ((rho u)^n + (rho u)^n+1)/2 g)."""
    nx, ny, nz, dx, g = 5, 4, 6, 0.1, -0.7
    grav = _const_z_table(nz, dx, lambda z: g, lambda z: 0.0, lambda z: 0.0)
    o = ob.Oracle(nx, ny, nz, dx, G, (P,) * 6, grav)
    rho, p = 1.3, 0.9
    g = float(np.float32(g))                      # the fp32 table node the oracle sees
    o.set_state(_fields((nz, ny, nx), rho, u0, p, 0.4))
    c0 = o.reduce_conserved()
    t = 0.0
    for s, dt in enumerate((0.02, 0.013, 0.031, 0.02)):
        o.step(dt, s % 6)
        t += dt
        f = o.get_state()
        uz = float(np.float32(u0[2])) + g * t
        assert np.max(np.abs(f[3] - uz)) <= 2e-15
        assert np.max(np.abs(f[0] - np.float32(rho))) <= 1e-15 and np.max(np.abs(f[4] - np.float32(p))) <= 2e-15
        assert np.array_equal(f[1], np.full_like(f[1], np.float32(u0[0]))) and np.array_equal(f[2], np.full_like(f[2], np.float32(u0[1])))
        assert np.max(np.abs(f[5] - np.float32(0.4))) <= 1e-15 and np.max(np.abs(f[6:])) <= 1e-14
    c1 = o.reduce_conserved()
    vol = nx * ny * nz * dx ** 3
    r32 = float(np.float32(rho))
    dke = 0.5 * r32 * vol * ((float(np.float32(u0[2])) + g * t) ** 2 - float(np.float32(u0[2])) ** 2)
    assert c1[4] - c0[4] == pytest.approx(dke, abs=1e-14)
    assert c1[3] - c0[3] == pytest.approx(r32 * vol * g * t, abs=1e-15)
    assert c1[0] == pytest.approx(c0[0], abs=1e-16)


def test_entropy_wave_in_free_fall_keeps_the_velocity_uniform():
    """Equivalence principle: gas of NON-uniform density with uniform pressure and velocity in a uniform field falls as
    a whole — u = u0 + g t stays uniform while the density pattern is advected.  One sweep of the scheme reproduces
    this exactly (to round-off) precisely because the momentum source is centred in time on the density,
    dt (rho'^n + rho'^n+1)/2 g (H9), and the traced states carry the half-step velocity u + dt g/2 (H6):
    (rho u)^n+1 = rho^n u + (u + dt g/2)(rho^n+1 - rho^n) + dt g (rho^n + rho^n+1)/2 = rho^n+1 (u + dt g).
    The energy source dt ((rho u)^n + (rho u)^n+1)/2 g then leaves the pressure uniform up to the third-order
    remainder (gamma - 1)(dt g)^2 (rho^n+1 - rho^n)/8."""
    n, dx, g, dt, u0, p0 = 32, 1.0 / 32, -0.9, 0.4 / 32, 0.4, 0.9
    grav = _const_z_table(n, dx, lambda z: g, lambda z: 0.0, lambda z: 0.0)
    g = float(np.float32(g))
    z = (np.arange(n) + 0.5) * dx
    f = _fields((n, 1, 1), 1.0, (0.0, 0.0, u0), p0)
    f[0] = (1.0 + 0.3 * np.sin(2 * math.pi * z))[:, None, None]
    o = ob.Oracle(1, 1, n, dx, G, (P,) * 6, grav)
    o.set_state(f)
    o.sweep(2, dt)
    s = o.get_state()[:, :, 0, 0]
    drho = s[0] - f[0, :, 0, 0].astype(np.float64)
    assert np.max(np.abs(drho)) > 1e-3                                  # the density pattern really moved
    assert np.max(np.abs(s[3] - (float(np.float32(u0)) + g * dt))) <= 1e-15
    rem = (G - 1.0) * (dt * g) ** 2 * drho / 8.0
    assert np.max(np.abs(s[4] - float(np.float32(p0)) - rem)) <= 1e-15
    assert np.max(np.abs(rem)) > 1e-8


def test_free_fall_radial_pencil_through_the_centre_is_exact():
    """RADIAL table with constant g(r) = g0 and no base state, on a 1-D window of cells that all lie on one side of
    the centre on the line through it: r = |x - cx|, the acceleration is g0 (x - cx)/r = +g0 exactly (base_at:
    direction along X - centre), so the gas falls freely, exactly.  The mirror window on the other side falls the
    other way."""
    n, dx, g0 = 12, 0.05, -0.6
    tab = dict(kind=ob.GRAV_RADIAL, s0=0.0, ds=0.01, center=(0.0, 0.5 * dx, 0.5 * dx),
               g=np.full(400, g0, dtype=np.float32), rho0=np.zeros(400, dtype=np.float32), p0=np.zeros(400, dtype=np.float32))
    for side in (+1, -1):
        org = (3, 0, 0) if side > 0 else (-3 - n, 0, 0)
        o = ob.Oracle(n, 1, 1, dx, G, (O, O, P, P, P, P), tab, org=org)
        o.set_state(_fields((1, 1, n), 1.1, (0.0, 0.0, 0.0), 0.8))
        t = 0.0
        for s in range(3):
            o.step(0.01, s)
            t += 0.01
        f = o.get_state()
        assert np.max(np.abs(f[1] - side * float(np.float32(g0)) * t)) <= 1e-16
        assert not f[2].any() and not f[3].any()
        assert np.max(np.abs(f[0] - np.float32(1.1))) <= 1e-15


def test_radial_field_direction_and_table_argument_from_one_small_step():
    """Harmonic field g(r) = -3 r (linear in r: reproduced exactly by the table's linear interpolation), uniform gas
    at rest, centre off the grid nodes.  After one step that is tiny against dx / c the pressure response is
    O(dt^2), so every cell has du = dt g(r) (X - centre)/r = -3 dt (X - centre), component by component."""
    n, dx = 10, 0.1
    cen = (0.43, 0.57, 0.36)
    nodes = 300
    ds = 0.005
    r = ds * np.arange(nodes)
    tab = dict(kind=ob.GRAV_RADIAL, s0=0.0, ds=ds, center=cen, g=(-3.0 * r).astype(np.float32),
               rho0=np.zeros(nodes, dtype=np.float32), p0=np.zeros(nodes, dtype=np.float32))
    o = ob.Oracle(n, n, n, dx, G, (P,) * 6, tab)
    o.set_state(_fields((n, n, n), 1.0, (0.0, 0.0, 0.0), 0.6))
    dt = 1e-6 * dx
    o.step(dt, 0)
    f = o.get_state()
    x = (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    g32 = (-3.0 * r).astype(np.float32).astype(np.float64)      # the fp32 table nodes the oracle sees
    rr = np.sqrt((X - cen[0]) ** 2 + (Y - cen[1]) ** 2 + (Z - cen[2]) ** 2)
    gr = np.interp(rr, r, g32)
    for d, XX in enumerate((X, Y, Z)):
        exp = dt * gr * (XX - cen[d]) / rr
        assert np.max(np.abs(f[1 + d] - exp)) <= 1e-6 * np.max(np.abs(exp))
    assert np.max(np.abs(f[1])) > 0.3 * 3.0 * dt * 0.4          # ... and it is not trivially zero


# ---------------------------------------------------------------- (b) split invariance --------------------------------
def _isothermal_column(n, frac, amp=0.05, t_end=0.25, cfl=0.4, nxy=1):
    """1-D isothermal atmosphere (rho0 = exp(-z/H), p0 = H rho0, g = -1; H = 0.6) between reflecting walls with the
    velocity pulse u_z = amp sin(pi z) on top, carried with the table (frac rho0, frac p0, g) — hydrostatic for every
    frac — and the rest of the state in rho', p'.  Returns the full state at t_end (fixed dt: same for every frac)."""
    H, dx = 0.6, 1.0 / n
    grav = _const_z_table(n, dx, lambda z: -1.0, lambda z: frac * np.exp(-z / H), lambda z: frac * H * np.exp(-z / H),
                          z_of_node=lambda z: np.abs(z))           # nodes behind the lower wall: unused (images), keep them finite
    z = (np.arange(n) + 0.5) * dx
    # cell means of the exact profile, so that both splits start from the same smooth data
    rho = H * (np.exp(-(z - 0.5 * dx) / H) - np.exp(-(z + 0.5 * dx) / H)) / dx
    f = np.zeros((15, n, nxy, nxy), dtype=np.float32)
    f[0] = rho[:, None, None]
    f[4] = (H * rho)[:, None, None]
    f[3] = (amp * np.sin(math.pi * z))[:, None, None]
    f[5] = 0.5
    o = ob.Oracle(nxy, nxy, n, dx, G, (P, P, P, P, R, R), grav)
    o.set_state(f)
    steps = int(math.ceil(t_end / (cfl * dx / (math.sqrt(G * H) + amp))))
    dt = t_end / steps
    for s in range(steps):
        o.sweep(2, dt)
    return o.get_state()[:, :, 0, 0]


@pytest.mark.parametrize("amp,ns", [(0.05, (32, 64, 128)), (0.2, (64, 128, 256))])
def test_split_invariance_of_the_base_state_to_truncation_order(amp, ns):
    """the perturbation form is "valid for perturbations of any size".  The SAME physical state is
    advanced once with the whole hydrostatic profile in the table (rho', p' small) and once with only half of it in
    the table and the other half carried in rho', p' (a perturbation of order one, itself hydrostatic).  The two runs
    discretise the same equations, so they agree to truncation order: the difference falls like dx^2 under
    refinement.  A wrong sign or factor in the half-step sources -u d(rho0)/dx, -u d(p0)/dx, g rho'/rho of the
    tracing (H6), or a source of H9 that is not time centred, leaves a first-order difference (ratio 2 per doubling);
    the Mach 0.25 pulse (amp = 0.2) makes the terms that are quadratic in the velocity visible."""
    d = []
    for n in ns:
        a, b = _isothermal_column(n, 1.0, amp=amp), _isothermal_column(n, 0.5, amp=amp)
        d.append([np.mean(np.abs(a[k] - b[k])) for k in (0, 3, 4)])
    d = np.array(d)
    # the flow really moved and the splits really differ in storage
    assert np.max(np.abs(_isothermal_column(ns[0], 1.0, amp=amp)[3])) > 0.2 * amp
    assert np.all(d[0] > 1e-9)
    assert np.all(d[0] / d[1] > 3.6) and np.all(d[1] / d[2] > 3.8), d
    # ... and it is small in absolute terms already on the coarsest grid (the half split carries an O(1) hydrostatic
    # profile numerically)
    assert d[0][1] < 1e-3


def test_split_invariance_zero_table_limit():
    """frac = 0: no base state at all (the scheme is then plain PPM with a rho g source) — still the same physics."""
    d = []
    for n in (32, 64, 128):
        a, b = _isothermal_column(n, 1.0), _isothermal_column(n, 0.0)
        d.append([np.mean(np.abs(a[k] - b[k])) for k in (0, 3, 4)])
    d = np.array(d)
    assert np.all(d[0] / d[1] > 3.5) and np.all(d[1] / d[2] > 3.5), d


# ---------------------------------------------------------------- (c) energy budget -----------------------------------
def _bubble_box(n, t_end=1.0, cfl=0.5):
    """closed reflecting box, constant g = -1 along z, isothermal base state, a dense blob released from rest;
    returns (mass, E + potential energy, kinetic energy) before and after."""
    H, dx = 0.6, 1.0 / n
    grav = _const_z_table(n, dx, lambda z: -1.0, lambda z: np.exp(-np.abs(z) / H), lambda z: H * np.exp(-np.abs(z) / H))
    x = (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    rho0 = np.exp(-Z / H)
    blob = 1.0 + 0.5 * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.6) ** 2) / 0.15 ** 2)
    f = np.zeros((15, n, n, n), dtype=np.float32)
    f[0], f[4], f[5] = rho0 * blob, H * rho0, 0.5
    o = ob.Oracle(n, n, n, dx, G, (R,) * 6, grav)
    o.set_state(f)

    def budget():
        s = o.get_state()
        dv = dx ** 3
        ke = 0.5 * np.sum(s[0] * (s[1] ** 2 + s[2] ** 2 + s[3] ** 2)) * dv
        pe = np.sum(s[0] * Z) * dv                      # Phi = -g z = z
        c = o.reduce_conserved()
        return c[0], c[4] + pe, ke, pe
    b0 = budget()
    steps = int(math.ceil(t_end / (cfl * dx / (math.sqrt(G * H) + 0.3))))
    dt = t_end / steps
    for s in range(steps):
        o.step(dt, 0 if s % 2 == 0 else 5)
    return b0, budget()


def test_energy_budget_in_a_closed_box_with_gravity():
    """sum (E + rho Phi) dV is conserved by the equations; the scheme's momentum and energy sources are time centred
    (H9), so its drift is a truncation error that falls under refinement, and it is tiny against the energy that
    actually changes hands (potential -> kinetic + internal).  Mass is conserved to round-off (walls: no mass flux;
    pins the odd image of g behind the walls together with test (d))."""
    drift = []
    for n in (16, 32):
        b0, b1 = _bubble_box(n)
        assert abs(b1[0] - b0[0]) <= 1e-13 * b0[0]
        exch = abs(b1[3] - b0[3])                       # potential energy released
        assert b1[2] > 1e-4 and exch > 5e-4             # the blob really sank
        drift.append(abs(b1[1] - b0[1]) / exch)
    assert drift[0] < 5e-3 and drift[1] < 1.5e-3, drift       # a wrong sign / factor 2 in the energy source gives O(1)
    assert drift[0] / drift[1] > 2.5, drift


# ---------------------------------------------------------------- (d) mirror sign of g --------------------------------
def test_reflecting_walls_equal_the_doubled_periodic_run_with_odd_gravity():
    """C1/C3: ghost cells behind a reflecting wall take the base state of their mirror-image position, rho0 and p0
    even, the normal acceleration ODD.  So a box with reflecting z walls must evolve exactly like the upper half of a
    periodic box of twice the height holding the even extension of the state (u_z and the z-odd FV coefficients odd)
    under the table (rho0(|z|), p0(|z|), g sign(z))."""
    rng = np.random.default_rng(17)
    nx, ny, nz, dx, H = 6, 5, 8, 0.125, 0.7
    f = np.zeros((15, nz, ny, nx), dtype=np.float32)
    z = (np.arange(nz) + 0.5) * dx
    rho0 = np.exp(-z / H)
    f[0] = rho0[:, None, None] * (1.0 + 0.2 * rng.random((nz, ny, nx)))
    f[1:4] = 0.2 * rng.normal(size=(3, nz, ny, nx))
    f[4] = (H * rho0)[:, None, None] * (1.0 + 0.2 * rng.random((nz, ny, nx)))
    f[5] = 0.2 + 0.6 * rng.random((nz, ny, nx))
    f[6:] = 0.02 * rng.normal(size=(9, nz, ny, nx))
    gfun = lambda s: -0.8 * (1.0 + 0.3 * np.abs(s))
    ga = _const_z_table(nz, dx, gfun, lambda s: np.exp(-np.abs(s) / H), lambda s: H * np.exp(-np.abs(s) / H))
    a = ob.Oracle(nx, ny, nz, dx, G, (P, P, P, P, R, R), ga)
    a.set_state(f)
    # doubled box: z' in [0, 2L), the original sits in the upper half (z = z' - L), its mirror image in the lower half
    L = nz * dx
    # height above the lower wall of the original box that z' maps to (periodic beyond [0, 2L)), and the side it is on
    fold = lambda s: np.where(np.abs(s - L) <= L, np.abs(s - L), 2 * L - np.abs(s - L))
    sign = lambda s: np.where(np.abs(s - L) <= L, np.sign(s - L), -np.sign(s - L))
    gb = _const_z_table(2 * nz, dx, lambda s: gfun(fold(s)) * sign(s), lambda s: np.exp(-fold(s) / H), lambda s: H * np.exp(-fold(s) / H))
    low = f[:, ::-1].copy()
    low[3] *= -1.0
    for k in (8, 13, 14):           # m001, m101, m011: odd in z
        low[k] *= -1.0
    b = ob.Oracle(nx, ny, 2 * nz, dx, G, (P,) * 6, gb)
    b.set_state(np.concatenate([low, f], axis=1))
    m0 = a.reduce_conserved()[0]
    for s, dt in enumerate((0.02, 0.015, 0.02)):
        a.step(dt, 2 * s)
        b.step(dt, 2 * s)
    fa, fb = a.get_state(), b.get_state()
    assert np.max(np.abs(fa - fb[:, nz:])) <= 1e-13
    assert np.abs(fa[3]).max() > 0.05
    assert abs(a.reduce_conserved()[0] - m0) <= 1e-14 * m0          # no mass leaves through the walls


# ---------------------------------------------------------------- (e) table lookup off the nodes ----------------------
def test_table_lookup_reproduces_a_linear_table_exactly_off_the_nodes():
    """C1: point values of the base state are LINEAR interpolations between table nodes.  A table that is linear in s
    (nodes exactly representable in fp32) is therefore reproduced exactly at arbitrary r — also past the last node,
    where the last interval is extended — which a swapped weight, an off-by-one node or a wrong node spacing breaks."""
    n, dx = 9, 0.11
    cen = (0.31, 0.77, 0.52)
    nodes, ds = 33, 0.03125
    s = ds * np.arange(nodes)
    a_r, b_r, a_p, b_p = 2.0, -0.75, 1.5, 0.25
    tab = dict(kind=ob.GRAV_RADIAL, s0=0.0, ds=ds, center=cen, g=np.zeros(nodes, dtype=np.float32),
               rho0=(a_r + b_r * s).astype(np.float32), p0=(a_p + b_p * s).astype(np.float32))
    assert np.array_equal(tab["rho0"].astype(np.float64), a_r + b_r * s)        # exactly representable nodes
    o = ob.Oracle(n, n, n, dx, G, (P,) * 6, tab)
    f = _fields((n, n, n), 3.0, (0, 0, 0), 2.0)
    o.set_state(f)
    x = (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r = np.sqrt((X - cen[0]) ** 2 + (Y - cen[1]) ** 2 + (Z - cen[2]) ** 2)
    assert r.max() > s[-1] + 0.05 and r.min() < 0.1                             # cells beyond the table end, too
    assert np.max(np.abs(o.raw_field(0) - (3.0 - (a_r + b_r * r)))) <= 2e-15
    assert np.max(np.abs(o.raw_field(4) - (2.0 - (a_p + b_p * r)))) <= 2e-15
    assert np.max(np.abs(o.get_state()[0] - 3.0)) <= 1e-15
