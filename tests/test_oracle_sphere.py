"""Pins of the oracle's confining-sphere mode and rotation spin-up ("our star is
enclosed in an impenetrable and immovable sphere that is inscribed in the cubical domain ... a very simple boundary
condition at the sphere"; "adding a solid body rotational flow component ... gradually over the first several thousand
time steps").  Readings R23 / R24 in DESIGN.md.  Expected values come from the mathematics of the reading only:

  * a state at rest stays at rest bit for bit, solid cells are never touched;
  * the sphere is impenetrable: mass and tracked mass of the fluid cells are conserved to round-off in a violent flow;
  * a sphere that contains the whole grid is the plain reflecting box, bit for bit;
  * a pencil cut by the sphere is a 1-D reflecting box of the segment's length (against the oracle's plain REFLECT
    walls on a grid of that length, base state included), also for segments shorter than the four ghost cells (against
    the doubled periodic box, whose images wrap more than once);
  * swapping the x and y axes of the data swaps them in the result (the mask has the cube's symmetries);
  * the spin-up increment is du = domega e_z x (X - centre) exactly, so N increments give solid-body rotation and the
    angular momentum grows by domega times the moment of inertia.
"""
import numpy as np
import pytest

from oracle import binding as ob
from paper_1810_13416_b200 import workloads as W

P, R, O = ob.BC_PERIODIC, ob.BC_REFLECT, ob.BC_OPEN
G = 5.0 / 3.0


def _random_state(rng, shape, vel=0.3):
    f = np.zeros((15,) + shape, dtype=np.float32)
    f[0] = 1.0 + 0.3 * rng.random(shape)
    f[1:4] = vel * rng.normal(size=(3,) + shape)
    f[4] = 0.8 + 0.3 * rng.random(shape)
    f[5] = 0.2 + 0.6 * rng.random(shape)
    f[6:] = 0.02 * rng.normal(size=(9,) + shape)
    return f


def test_mask_is_the_inscribed_sphere_and_rejects_periodic_faces():
    n = 16
    o = ob.Oracle(n, n, n, 1.0 / n, G, (R,) * 6)
    o.set_sphere(0.5, (0.5, 0.5, 0.5))
    m = o.solid_mask()
    x = (np.arange(n) + 0.5) / n - 0.5
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    assert np.array_equal(m, X * X + Y * Y + Z * Z > 0.25)
    assert 0.45 < m.mean() < 0.50                       # 1 - pi/6 of the cube is outside
    assert not m[n // 2, n // 2, :].any()               # the pencils through the centre reach the cube faces
    with pytest.raises(ValueError):
        ob.Oracle(n, n, n, 1.0 / n, G, (P, P, R, R, R, R)).set_sphere(0.5, (0.5, 0.5, 0.5))


def test_state_at_rest_is_preserved_bitwise_and_solid_cells_are_never_touched():
    rng = np.random.default_rng(2)
    n = 12
    for cfg in (None, 4):
        if cfg is None:
            o = ob.Oracle(n, n, n, 1.0 / n, G, (R,) * 6)
            f = np.zeros((15, n, n, n), dtype=np.float32)
            f[0], f[4], f[5] = 1.3, 0.9, 0.4
        else:                                           # the hydrostatic convection-zone profile of configs 4/5
            w = W.make(4, n=n)
            o = ob.Oracle(n, n, n, w.dx, w.gamma, w.bc, w.grav)
            f = w.fields().numpy()
            f[1:4] = 0.0
        o.set_sphere(0.5, (0.5, 0.5, 0.5))
        m = o.solid_mask()
        f[:, m] = rng.random((15, int(m.sum()))).astype(np.float32) + 0.5       # junk in the solid cells: nothing may read it
        o.set_state(f)
        if cfg is not None:
            for k in (0, 4):
                o.raw_field(k)[~m] = 0.0                # exactly zero perturbation in the fluid
        ref = [o.raw_field(k).copy() for k in range(15)]
        for s in range(3):
            o.step(0.5 / n, s)
        for k in range(15):
            got = o.raw_field(k)
            assert np.array_equal(got[m], ref[k][m])                            # solid: untouched
            if cfg is not None:
                # hydrostatic star: p is rebuilt from E = p/(gamma-1), i.e. preserved to the last bit only, and that
                # 1e-16 noise then evolves (as in the cube: test_hydrostatic_base_state_preserved_bitwise...)
                # (the higher FV coefficients of the under-resolved r = 0.45 edge are rescaled by the P2 pre-limiter even
                # at rest: by design, in the cube as well — only the cell means m000 are checked)
                if k <= 5:
                    assert np.max(np.abs(got[~m] - ref[k][~m])) <= 1e-14
            elif k in (1, 2, 3):
                assert not got[~m].any()                                        # fluid: still at rest, exactly
            elif k == 4:
                assert np.max(np.abs(got[~m] - ref[k][~m])) <= 4e-16            # p goes through E: last-bit noise
            elif k in (0, 5):
                assert np.array_equal(got[~m], ref[k][~m])


def test_sphere_is_impenetrable_mass_and_tracked_mass_conserved_in_a_violent_flow():
    rng = np.random.default_rng(3)
    n = 14
    o = ob.Oracle(n, n, n, 1.0 / n, G, (R,) * 6)
    o.set_sphere(0.47, (0.5, 0.52, 0.48))               # off-centre, not touching every face
    f = _random_state(rng, (n, n, n), vel=0.6)
    o.set_state(f)
    c0 = o.reduce_conserved()
    m = o.solid_mask()
    full0 = o.get_state()
    assert c0[0] == pytest.approx(full0[0][~m].sum() / n ** 3, rel=1e-14)       # the sums run over the fluid cells only
    for s in range(5):
        o.step(o.cfl_dt(0.8), s)
    c1 = o.reduce_conserved()
    assert abs(c1[0] - c0[0]) <= 2e-14 * c0[0] and abs(c1[5] - c0[5]) <= 2e-14 * c0[5]
    assert abs(c1[4] - c0[4]) <= 2e-14 * c0[4]          # immovable walls do no work (g = 0)
    full1 = o.get_state()
    assert np.array_equal(full1[:, m], full0[:, m])
    assert np.abs(full1[0][~m] - full0[0][~m]).max() > 0.05                     # ... and the fluid really moved
    assert full1[5][~m].min() >= 0.0 and full1[5][~m].max() <= 1.0


def test_a_sphere_that_contains_the_grid_is_the_reflecting_box_bitwise():
    rng = np.random.default_rng(4)
    nx, ny, nz = 9, 7, 8
    f = _random_state(rng, (nz, ny, nx))
    res = []
    for sph in (False, True):
        o = ob.Oracle(nx, ny, nz, 0.1, G, (R,) * 6)
        if sph:
            o.set_sphere(5.0, (0.4, 0.3, 0.4))
            assert not o.solid_mask().any()
        o.set_state(f)
        for s in range(3):
            o.step(0.02, 2 * s)
        res.append(o.get_state())
    assert np.array_equal(res[0], res[1])


@pytest.mark.parametrize("seg", [(5, 14), (3, 5), (7, 8), (6, 6)])
def test_pencil_cut_by_the_sphere_is_a_1d_reflecting_box_of_the_segment(seg):
    """1-D grid of 20 cells, sphere = the interval that leaves cells lo..hi fluid.  Its evolution must equal (a) for
    segments of >= 4 cells the oracle's plain REFLECT box of that many cells placed at the same global position (base
    state included), and (b) for ANY length the doubled periodic box with the even extension of the data — whose
    periodic images wrap as often as needed (fewer cells than ghosts)."""
    rng = np.random.default_rng(5)
    n, dx = 20, 0.05
    lo, hi = seg
    L = hi - lo + 1
    cen = ((lo + hi + 1) * 0.5 * dx, 0.5 * dx, 0.5 * dx)
    rad = (L * 0.5 - 0.25) * dx if L > 1 else 0.3 * dx
    z = dx * np.arange(-8, 2 * n + 9) * 0.5
    grav = None
    f = _random_state(rng, (1, 1, n), vel=0.2)
    a = ob.Oracle(n, 1, 1, dx, G, (R,) * 6, grav)
    a.set_sphere(rad, cen)
    m = a.solid_mask()[0, 0]
    assert np.array_equal(np.nonzero(~m)[0], np.arange(lo, hi + 1))
    a.set_state(f)
    dts = (0.004, 0.003, 0.004, 0.002)
    for dt in dts:
        a.sweep(0, dt)
    got = a.get_state()[:, 0, 0, lo:hi + 1]
    if L >= 4:
        b = ob.Oracle(L, 1, 1, dx, G, (R,) * 6, grav, org=(lo, 0, 0))
        b.set_state(f[:, :, :, lo:hi + 1])
        for dt in dts:
            b.sweep(0, dt)
        assert np.array_equal(got, b.get_state()[:, 0, 0, :])
    fl = f[:, :, :, lo:hi + 1]
    mir = fl[:, :, :, ::-1].copy()
    mir[1] *= -1.0
    for k in (6, 12, 13):                               # m100, m110, m101: odd in x
        mir[k] *= -1.0
    c = ob.Oracle(2 * L, 1, 1, dx, G, (P,) * 6, None)
    c.set_state(np.concatenate([mir, fl], axis=3))
    for dt in dts:
        c.sweep(0, dt)
    assert np.max(np.abs(got - c.get_state()[:, 0, 0, L:])) <= 1e-13
    assert np.abs(got[1]).max() > 0 or L == 1


def test_pencil_segment_uses_the_base_state_of_the_mirror_image_position():
    """the same 1-D comparison with the stratified RADIAL base state of configs 4/5 switched on: the segment's ghost cells
    must take rho0, p0 at their mirror-image positions and the radial g with the sign flipped"""
    rng = np.random.default_rng(6)
    w = W.make(4, n=32)
    n, dx = 32, w.dx
    cy = (16 + 0.5) * dx                                # the pencil y = z = 16 passes half a cell from the centre
    lo, hi = 6, 25
    rad = np.sqrt((10.0 * dx - 0.25 * dx) ** 2 + 2 * (cy - 0.5) ** 2)
    f = w.fields((0, 16, 16), (n, 17, 17)).numpy()
    f[1] = 0.05 * rng.normal(size=f[1].shape).astype(np.float32)
    a = ob.Oracle(n, 1, 1, dx, w.gamma, (R,) * 6, w.grav, org=(0, 16, 16))
    a.set_sphere(rad, (0.5, 0.5, 0.5))
    assert np.array_equal(np.nonzero(~a.solid_mask()[0, 0])[0], np.arange(lo, hi + 1))
    b = ob.Oracle(hi - lo + 1, 1, 1, dx, w.gamma, (R,) * 6, w.grav, org=(lo, 16, 16))
    a.set_state(f)
    b.set_state(f[:, :, :, lo:hi + 1])
    for s in range(4):
        a.sweep(0, 0.4 * dx)
        b.sweep(0, 0.4 * dx)
    assert np.array_equal(a.get_state()[:, 0, 0, lo:hi + 1], b.get_state()[:, 0, 0, :])
    assert np.abs(b.get_state()[0, 0, 0] - f[0, 0, 0, lo:hi + 1]).max() > 1e-4


def test_axis_swap_symmetry_with_the_sphere():
    rng = np.random.default_rng(7)
    n = 10
    f = _random_state(rng, (n, n, n))
    o = ob.Oracle(n, n, n, 0.1, G, (R,) * 6)
    o.set_sphere(0.46, (0.5, 0.5, 0.5))
    o.set_state(f)
    o.step(0.02, 0)                                     # xyz
    ref = o.get_state()
    # swap x <-> y: fields ux <-> uy, m100 <-> m010, m200 <-> m020, m101 <-> m011; arrays transposed in (y, x)
    perm = [0, 2, 1, 3, 4, 5, 7, 6, 8, 10, 9, 11, 12, 14, 13]
    sw = lambda a: np.ascontiguousarray(np.transpose(a[perm], (0, 1, 3, 2)))
    o2 = ob.Oracle(n, n, n, 0.1, G, (R,) * 6)
    o2.set_sphere(0.46, (0.5, 0.5, 0.5))
    o2.set_state(sw(f))
    o2.step(0.02, 2)                                    # yxz
    assert np.max(np.abs(o2.get_state() - sw(ref))) <= 1e-13


def test_spin_up_increment_is_solid_body_rotation_about_the_centre():
    rng = np.random.default_rng(8)
    n = 12
    dx = 1.0 / n
    o = ob.Oracle(n, n, n, dx, G, (R,) * 6)
    cen = (0.5, 0.5, 0.5)
    o.set_sphere(0.5, cen)
    f = _random_state(rng, (n, n, n))
    o.set_state(f)
    m = o.solid_mask()
    full0 = o.get_state()
    x = (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    lz = lambda s: np.sum((s[0] * ((X - 0.5) * s[2] - (Y - 0.5) * s[1]))[~m])
    inertia = np.sum((full0[0] * ((X - 0.5) ** 2 + (Y - 0.5) ** 2))[~m])
    nramp, omega = 25, 0.8
    for _ in range(nramp):
        o.spin_up(omega / nramp)
    s = o.get_state()
    assert np.max(np.abs((s[1] - full0[1] + omega * (Y - 0.5))[~m])) <= 1e-14
    assert np.max(np.abs((s[2] - full0[2] - omega * (X - 0.5))[~m])) <= 1e-14
    assert np.array_equal(s[3], full0[3]) and np.array_equal(s[0], full0[0]) and np.array_equal(s[4], full0[4])
    assert np.array_equal(s[:, m], full0[:, m])                                  # the solid cells do not rotate
    assert lz(s) - lz(full0) == pytest.approx(omega * inertia, rel=1e-12)
