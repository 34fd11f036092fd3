"""How far does reading R8' (switch-free characteristic tracing) move the SOLUTION from the
hard-switched tracing of Colella & Woodward 1984, the only source the paper names for this step (PAPER.md L87 ->
ref. [30], L189)?

R8' is identical to the textbook form only where all three characteristics point at the face (supersonic flow).  In
subsonic flow — all of configs 1, 2, 4, 5 — the acoustic family that LEAVES the face contributes its edge-value
amplitude, which the textbook form drops.  The Riemann problem takes the C+ invariant from its left state and the
C- invariant from its right state, and R8' leaves exactly those unchanged, so the two schemes differ only through
terms that are quadratic in the wave amplitude.  These tests quantify that with tests/cw84_comparator.py (a test-only
numpy 1-D PPM with both tracings):

  * the comparator's "r8p" mode reproduces the oracle's sweep to round-off (so the comparison is about H6 only);
  * smooth subsonic flow: |R8' - CW84| = O(dx^2), a few per cent of either scheme's own truncation error, and both
    have the same order and error constant against a fine-grid reference;
  * Sod shock tube: both stay in the same first-order L1 band about the exact solution.
"""
import numpy as np

from oracle import binding as ob

import cw84_comparator as cw
import exact_riemann as ex

G = 5.0 / 3.0
P, R = ob.BC_PERIODIC, ob.BC_REFLECT


def _f32(a):
    return np.asarray(a, dtype=np.float32).astype(np.float64)


def _oracle_run(rho, u, p, gamma, dts, bc):
    n = rho.size
    b = (R, R) if bc == "reflect" else (P, P)
    o = ob.Oracle(n, 1, 1, 1.0 / n, gamma, b + (P, P, P, P))
    f = np.zeros((15, 1, 1, n), dtype=np.float32)
    f[0, 0, 0], f[1, 0, 0], f[4, 0, 0], f[5] = rho, u, p, 0.5
    o.set_state(f)
    for dt in dts:
        o.sweep(0, dt)
    s = o.get_state()[:, 0, 0, :]
    return s[0], s[1], s[4]


def _smooth(n):
    """subsonic (Mach 0.2-0.3) superposition of an entropy wave and acoustic waves of both families"""
    x = (np.arange(n) + 0.5) / n
    return (_f32(1 + 0.2 * np.sin(2 * np.pi * x)), _f32(0.3 + 0.1 * np.sin(2 * np.pi * x + 1.0)),
            _f32(1 + 0.1 * np.cos(2 * np.pi * x)))


def _sod(n):
    x = (np.arange(n) + 0.5) / n
    left = x < 0.5
    return x, _f32(np.where(left, 1.0, 0.125)), np.zeros(n), _f32(np.where(left, 1.0, 0.1))


def test_comparator_in_r8prime_mode_is_the_oracle():
    rho, u, p = _smooth(48)
    a = cw.run(rho, u, p, G, 0.3, 0.8, "periodic", "r8p")
    o = _oracle_run(rho, u, p, G, a[3], "periodic")
    assert max(np.abs(a[k] - o[k]).max() for k in range(3)) < 1e-13
    x, rho, u, p = _sod(100)
    a = cw.run(rho, u, p, 1.4, 0.2, 0.8, "reflect", "r8p")
    o = _oracle_run(rho, u, p, 1.4, a[3], "reflect")
    assert max(np.abs(a[k] - o[k]).max() for k in range(3)) < 1e-12
    # ... and its "cw84" mode really is a different scheme in subsonic flow
    b = cw.run(rho, u, p, 1.4, 0.2, 0.8, "reflect", "cw84", dts=a[3])
    assert np.abs(a[0] - b[0]).max() > 1e-4


def test_r8prime_differs_from_cw84_by_second_order_terms_in_smooth_subsonic_flow():
    fine = _smooth(2048)
    ref = cw.run(*fine, G, 0.3, 0.8, "periodic", "r8p")
    diff, err_a, err_b = [], [], []
    for n in (32, 64, 128):
        rho, u, p = _smooth(n)
        a = cw.run(rho, u, p, G, 0.3, 0.8, "periodic", "r8p")
        b = cw.run(rho, u, p, G, 0.3, 0.8, "periodic", "cw84", dts=a[3])
        diff.append(max(np.mean(np.abs(a[k] - b[k])) for k in range(3)))
        rr = ref[0].reshape(n, -1).mean(axis=1)
        err_a.append(np.mean(np.abs(a[0] - rr)))
        err_b.append(np.mean(np.abs(b[0] - rr)))
    # the two schemes converge to each other like dx^2 ...
    assert diff[0] / diff[1] > 3.6 and diff[1] / diff[2] > 3.6, diff
    # ... the difference is a small fraction of either scheme's own truncation error ...
    assert all(d < 0.06 * e for d, e in zip(diff, err_a)), (diff, err_a)
    # ... and both have the same order and the same error constant (within 3 per cent)
    for ea, eb in zip(err_a, err_b):
        assert abs(ea - eb) < 0.03 * ea
    assert err_a[0] / err_a[1] > 3.6 and err_b[0] / err_b[1] > 3.6


def test_r8prime_and_cw84_stay_in_the_same_first_order_band_on_sod():
    ea, eb, dab = [], [], []
    for n in (100, 200, 400):
        x, rho, u, p = _sod(n)
        a = cw.run(rho, u, p, 1.4, 0.2, 0.8, "reflect", "r8p")
        b = cw.run(rho, u, p, 1.4, 0.2, 0.8, "reflect", "cw84")
        exact = ex.profile(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4, x, 0.5, 0.2)
        ea.append(np.mean(np.abs(a[0] - exact[:, 0])))
        eb.append(np.mean(np.abs(b[0] - exact[:, 0])))
        dab.append(np.mean(np.abs(a[0] - b[0])))
    for k in range(3):
        assert abs(ea[k] - eb[k]) < 0.03 * eb[k]            # same L1 error about the exact solution within 3 per cent
        assert dab[k] < 0.08 * eb[k]                        # and closer to each other than to the exact solution by > 10x
    assert ea[0] / ea[1] > 1.6 and eb[0] / eb[1] > 1.6      # both first order in L1
