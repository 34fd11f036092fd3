"""Pins of the oracle's 1-D routines against what the mathematics fixes.

None of these re-types the oracle's formula: each compares with a closed form, a hand-computed
value, brute-force quadrature, or a textbook exact solver (tests/exact_riemann.py).
"""
import math

import numpy as np
import pytest
from numpy.polynomial import Polynomial as Poly
from numpy.polynomial.legendre import leggauss

from oracle import binding as ob

import exact_riemann as ex

RNG = np.random.default_rng(7)


# ---------------------------------------------------------------- H1 ----------------
def _cell_avg(poly, j):
    P = poly.integ()
    return P(j + 0.5) - P(j - 0.5)


def test_h1_exact_for_cubic_cell_averages():
    for _ in range(20):
        c = RNG.normal(size=4)
        poly = Poly(c)
        av = [_cell_avg(poly, j) for j in (-1, 0, 1, 2)]
        assert ob.h1_face(*av) == pytest.approx(poly(0.5), abs=1e-13)


def test_h1_quartic_error_is_minus_four_fifths():
    poly = Poly([0, 0, 0, 0, 1.0])
    av = [_cell_avg(poly, j) for j in (-1, 0, 1, 2)]
    assert ob.h1_face(*av) - poly(0.5) == pytest.approx(-4.0 / 5.0, abs=1e-12)


# ---------------------------------------------------------------- H2 -------------------------------
def test_h2_constant_and_extremum():
    assert ob.h2_limit(2.0, 2.0, 2.0, 2.0, 2.0) == (2.0, 2.0)
    # local extremum: flat parabola
    assert ob.h2_limit(1.0, 3.0, 1.5, 2.0, 2.2) == (3.0, 3.0)


def test_h2_three_cw_cases_hand_values():
    # (a) monotone, no overshoot: faces kept.  q = 0,1,2, faces 0.5,1.5
    assert ob.h2_limit(0.0, 1.0, 2.0, 0.5, 1.5) == (0.5, 1.5)
    # (b) parabola overshoots near the right: qi close to qR: L <- 3 qi - 2 R
    # q = (0, 0.9, 1), faces 0.1, 1.0 : D = 0.9, q6 = 6 (0.9 - 0.55) = 2.1 -> D q6 = 1.89 > 0.81
    L, R = ob.h2_limit(0.0, 0.9, 1.0, 0.1, 1.0)
    assert (L, R) == pytest.approx((3 * 0.9 - 2 * 1.0, 1.0), abs=1e-15)
    # (c) mirrored: qi close to qL: R <- 3 qi - 2 L
    L, R = ob.h2_limit(0.0, 0.1, 1.0, 0.0, 0.9)
    assert (L, R) == pytest.approx((0.0, 3 * 0.1 - 2 * 0.0), abs=1e-15)
    # faces are first clipped to the neighbouring means
    L, R = ob.h2_limit(0.0, 1.0, 2.0, -0.3, 2.4)
    assert L >= 0.0 and R <= 2.0


def test_h2_monotone_data_no_new_extrema_and_symmetries():
    for _ in range(200):
        q = np.sort(RNG.normal(size=5))
        fl = ob.h1_face(*q[0:4])
        fr = ob.h1_face(*q[1:5])
        L, R = ob.h2_limit(q[1], q[2], q[3], fl, fr)
        # parabola through (L, R, mean q[2]) is monotone: interior extremum test |q6| <= |D|
        D, q6 = R - L, 6 * (q[2] - 0.5 * (L + R))
        assert abs(q6) <= abs(D) + 1e-12
        assert q[1] - 1e-12 <= L <= q[2] + 1e-12 and q[2] - 1e-12 <= R <= q[3] + 1e-12
        # mirror symmetry i -> -i
        L2, R2 = ob.h2_limit(q[3], q[2], q[1], fr, fl)
        assert (L2, R2) == pytest.approx((R, L), abs=1e-14)
        # sign symmetry q -> -q
        L3, R3 = ob.h2_limit(-q[1], -q[2], -q[3], -fl, -fr)
        assert (L3, R3) == pytest.approx((-L, -R), abs=1e-14)


# ---------------------------------------------------------------- H3 ----------------
def test_h3_quadratic_is_smooth():
    for _ in range(20):
        a, b, c = RNG.normal(size=3)
        q = [a + b * j + c * j * j for j in range(-2, 3)]
        assert ob.h3_S(q) == pytest.approx(0.0, abs=1e-12)
        assert ob.h3_omega(ob.h3_S(q)) == 0.0


def test_h3_unit_step_hand_values():
    q = np.array([0.0] * 6 + [1.0] * 6)     # step between cells 5 and 6
    S = [ob.h3_S(q[j - 2:j + 3]) for j in range(2, 10)]
    # cells j-1=4, j=5, j+1=6, j+2=7 (indices 2..5 of S)
    assert S[2] == pytest.approx(1.0) and S[5] == pytest.approx(1.0)
    assert S[3] == pytest.approx(1.0 / 3.0) and S[4] == pytest.approx(1.0 / 3.0)
    assert S[0] == 0.0 and S[7] == 0.0
    assert all(ob.h3_omega(s) == 1.0 for s in S[2:6])


def test_h3_sine_extremum_not_clipped_and_ramp():
    # a sine resolved with >= 8 cells stays in the smooth regime at its extrema
    # closed form for a sampled sine (d2_j = -4 sin^2(k/2) sin(theta_j)):
    #   S = |2 cos(theta) sin(k)| / (|sin(theta-k)| + 2 |sin(theta)| + |sin(theta+k)|)
    for ncell in (8, 12, 16, 32):
        k = 2 * math.pi / ncell
        x = np.arange(-2, 3) * k
        for th in np.linspace(0.05, 2 * math.pi, 23):
            S = ob.h3_S(np.sin(x + th))
            cf = abs(2 * math.cos(th) * math.sin(k)) / (abs(math.sin(th - k)) + 2 * abs(math.sin(th)) + abs(math.sin(th + k)))
            assert S == pytest.approx(cf, abs=1e-9)
        # the cell that contains the extremum (|theta - pi/2| <= k/2): never limited for >= 12 cells per wave
        for off in np.linspace(-0.5, 0.5, 11):
            S = ob.h3_S(np.sin(x + math.pi / 2 + off * k))
            assert S <= (0.18 if ncell == 8 else 0.1)
            if ncell >= 12:
                assert ob.h3_omega(S) == 0.0
    x = np.arange(-2, 3) * 2 * math.pi / 16
    assert ob.h3_omega(ob.h3_S(np.cos(x))) == 0.0      # exactly at the extremum: symmetric -> S = 0
    assert ob.h3_omega(0.1) == 0.0 and ob.h3_omega(0.3) == pytest.approx(1.0)
    assert ob.h3_omega(0.2) == pytest.approx(0.5)


# ---------------------------------------------------------------- H4 -------------------------------
def test_h4_hand_values():
    g = 5.0 / 3.0
    # Mach-3 shock, pressure ratio 11, one intermediate cell: every ramp saturates -> 1
    p5 = [11.0, 11.0, 6.0, 1.0, 1.0]
    u2 = 0.75 * math.sqrt(g) * (3 - 1 / 3)
    assert ob.h4_ftilde(p5, u2, 0.0, math.sqrt(g * 6.0 / 2.0)) == pytest.approx(1.0)
    # weak jump |d1|/min p < 1/3 -> 0
    assert ob.h4_ftilde([1.2, 1.2, 1.1, 1.0, 1.0], 1.0, 0.0, 1.0) == 0.0
    # diverging flow -> 0
    assert ob.h4_ftilde(p5, 0.0, 1.0, 1.0) == 0.0
    # broad linear ramp: |d1|/|d2| = 0.5 < 0.75 -> 0
    assert ob.h4_ftilde([9.0, 7.0, 5.0, 3.0, 1.0], 2.0, 0.0, 1.0) == 0.0
    # half-way values of each ramp, by hand: steep = 10 (0.8 - 0.75) = 0.5, jump = 3*0.8/1.2 - 1 = 1, conv = 0.02/0.05 = 0.4
    v = ob.h4_ftilde([2.2, 2.0, 1.6, 1.2, 1.2], 0.02, 0.0, 1.0)
    assert v == pytest.approx(0.5 * 1.0 * 0.4, rel=1e-12)


# ---------------------------------------------------------------- H5 -------------------------------
def _parabola(ql, qr, qi):
    dq, q6 = qr - ql, 6 * (qi - 0.5 * (ql + qr))
    x = Poly([0.5, 1.0])                        # x = xi + 1/2
    return ql + x * (dq + q6 * (1 - x))


def test_h5_matches_quadrature_of_the_parabola():
    for _ in range(50):
        ql, qr, qi = RNG.normal(size=3)
        par = _parabola(ql, qr, qi)
        P = par.integ()
        assert P(0.5) - P(-0.5) == pytest.approx(qi, abs=1e-13)
        for s in (0.0, 1e-3, 0.3, 0.8, 1.0):
            if s > 0:
                fp = (P(0.5) - P(0.5 - s)) / s
                fm = (P(-0.5 + s) - P(-0.5)) / s
            else:
                fp, fm = qr, ql
            assert ob.h5_Fplus(ql, qr, qi, s) == pytest.approx(fp, abs=1e-11)
            assert ob.h5_Fminus(ql, qr, qi, s) == pytest.approx(fm, abs=1e-11)
        assert ob.h5_Fplus(ql, qr, qi, 1.0) == pytest.approx(qi, abs=1e-14)
        assert ob.h5_Fminus(ql, qr, qi, 1.0) == pytest.approx(qi, abs=1e-14)


# ---------------------------------------------------------------- H6 -------------------------------
def test_h6_dt_to_zero_and_uniform():
    ql, qr, qi = RNG.normal(size=5), RNG.normal(size=5), RNG.normal(size=5)
    for u in (-3.0, -0.2, 0.2, 3.0):      # super/sub-sonic both ways (c = 1)
        qi2 = qi.copy()
        qi2[1] = u
        WL, WR = ob.h6_trace(ql, qr, qi2, 1.3, 1.0, 1e-13)
        assert WL == pytest.approx(qr, abs=1e-11) and WR == pytest.approx(ql, abs=1e-11)
    q = np.array([0.3, 0.7, -0.2, 0.1, 0.4])
    WL, WR = ob.h6_trace(q, q, q, 1.3, 1.1, 0.6)
    assert np.array_equal(WL, q) and np.array_equal(WR, q)


def test_h6_sources_added_to_both_states():
    q = np.array([0.3, 0.7, -0.2, 0.1, 0.4])
    WL, WR = ob.h6_trace(q, q, q, 1.3, 1.1, 0.6, src=(0.01, -0.02, 0.03))
    exp = q + np.array([0.01, -0.02, 0, 0, 0.03])
    assert WL == pytest.approx(exp, abs=1e-15) and WR == pytest.approx(exp, abs=1e-15)


def test_h6_entropy_wave_is_scalar_ppm_advection():
    # u, p uniform; rho varies: u_L = u, p_L = p, rho_L = average of rho over the u*dt domain
    for u in (0.4, -0.4):
        rl, rr, ri = 0.9, 1.2, 1.0
        ql = np.array([rl, u, 0.1, 0.2, 0.5])
        qr = np.array([rr, u, 0.1, 0.2, 0.5])
        qi = np.array([ri, u, 0.1, 0.2, 0.5])
        dtdx = 0.7
        WL, WR = ob.h6_trace(ql, qr, qi, 1.0, 1.0, dtdx)
        P = _parabola(rl, rr, ri).integ()
        s = abs(u) * dtdx
        assert WL[1] == pytest.approx(u, abs=1e-15) and WL[4] == pytest.approx(0.5, abs=1e-15)
        assert WR[1] == pytest.approx(u, abs=1e-15) and WR[4] == pytest.approx(0.5, abs=1e-15)
        if u > 0:
            assert WL[0] == pytest.approx((P(0.5) - P(0.5 - s)) / s, abs=1e-12)
            # the contact moves away from the left face: its amplitude there is the edge value
            # (zero-width domain of dependence; reading R8')
            assert WR[0] == pytest.approx(rl, abs=1e-12)
        else:
            assert WR[0] == pytest.approx((P(-0.5 + s) - P(-0.5)) / s, abs=1e-12)
            assert WL[0] == pytest.approx(rr, abs=1e-12)


def test_h6_is_continuous_across_the_sign_changes_of_the_characteristic_speeds():
    # reading R8': no hard switch on sign(lambda^k) -> traced states are continuous in u
    ql = np.array([0.9, 0.1, 0.3, -0.2, 0.8]); qr = np.array([1.2, -0.1, 0.1, 0.2, 1.1])
    for u0 in (0.0, 1.0, -1.0):          # contact, and the two sonic points (c = 1)
        outs = []
        for eps in (-1e-9, 1e-9):
            qi = 0.5 * (ql + qr) + np.array([0.02, 0, 0, 0, -0.03])
            qi[1] = u0 + eps
            outs.append(np.concatenate(ob.h6_trace(ql, qr, qi, 1.3, 1.0, 0.6)))
        assert np.max(np.abs(outs[0] - outs[1])) < 1e-8


def test_h6_acoustic_wave_uses_plus_characteristic_domain():
    # right-moving simple acoustic wave (linear): dp = rho c du, drho = dp / c^2; all three
    # families see linear profiles, and the left state must equal the average over the u+c domain.
    rho, c, u0 = 1.0, 1.0, 0.0
    du = 1e-6
    ql = np.array([-du, u0 - du, 0, 0, -du])     # (rho', u, v, w, p') linear across the cell
    qr = np.array([+du, u0 + du, 0, 0, +du])
    qi = 0.5 * (ql + qr)
    dtdx = 0.5
    WL, _ = ob.h6_trace(ql, qr, qi, rho, c, dtdx)
    sp = (u0 + c) * dtdx
    exp = du * (1 - sp)                              # average of a linear profile over [1/2 - sp, 1/2]
    assert WL[1] == pytest.approx(u0 + exp, rel=1e-9)
    assert WL[4] == pytest.approx(exp, rel=1e-9)


# ---------------------------------------------------------------- H7 -------------------------------
G = 5.0 / 3.0


def test_h7_equal_states_and_stationary_contact():
    s = np.array([1.3, 0.4, -0.1, 0.2, 0.9])
    out, ps, us = ob.h7_riemann(s, s, G)
    assert out == pytest.approx(s, abs=1e-14) and ps == pytest.approx(0.9) and us == pytest.approx(0.4)
    L = np.array([2.0, 0.0, 0.3, 0.0, 1.0])
    R = np.array([0.5, 0.0, -0.3, 0.0, 1.0])
    out, ps, us = ob.h7_riemann(L, R, G)
    assert ps == pytest.approx(1.0, abs=1e-15) and us == 0.0
    assert out[0] * out[1] == 0.0                          # no mass flux through a stationary contact


def test_h7_symmetric_collision_rankine_hugoniot_closed_form():
    rho, p = 1.0, 1.0
    for v in (0.05, 0.5, 2.0):
        A, B = 2.0 / ((G + 1) * rho), (G - 1) / (G + 1) * p
        x = (v * v + math.sqrt(v ** 4 + 4 * A * v * v * (p + B))) / (2 * A)
        out, ps, us = ob.h7_riemann([rho, v, 0, 0, p], [rho, -v, 0, 0, p], G)
        assert us == pytest.approx(0.0, abs=1e-15)
        assert ps == pytest.approx(p + x, rel=1e-9)


def test_h7_two_shock_cases_match_exact_solver():
    cases = [((1.0, 2.0, 1.0), (1.5, -1.0, 2.0)), ((1.0, 0.5, 0.4), (0.3, -2.5, 0.1)), ((5.0, 1.0, 3.0), (4.0, -1.5, 2.5)),
             ((1.0, 3.0, 1.0), (1.0, 1.0, 1.0))]
    for (rl, ul, pl), (rr, ur, pr) in cases:
        pe, ue = ex.star(rl, ul, pl, rr, ur, pr, G)
        assert pe > max(pl, pr)                 # both waves are shocks: the two-shock solver is exact
        out, ps, us = ob.h7_riemann([rl, ul, 0.7, -0.3, pl], [rr, ur, -0.7, 0.3, pr], G)
        assert ps == pytest.approx(pe, rel=1e-8) and us == pytest.approx(ue, abs=1e-8)
        re_, ue_, pe_ = ex.sample(rl, ul, pl, rr, ur, pr, G, 0.0)
        assert out[[0, 1, 4]] == pytest.approx([re_, ue_, pe_], rel=1e-7)
        # transverse velocities come from the upwind side of the contact
        assert (out[2], out[3]) == ((0.7, -0.3) if us >= 0 else (-0.7, 0.3))


def test_h7_sod_close_to_exact_and_acoustic_limit():
    g = 1.4
    pe, ue = ex.star(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
    _, ps, us = ob.h7_riemann([1.0, 0, 0, 0, 1.0], [0.125, 0, 0, 0, 0.1], g)
    assert abs(ps - pe) < 2e-3 * pe * 10 and abs(us - ue) < 2e-2      # rarefaction treated as a shock
    assert ps != pe
    # acoustic limit: error of the two-shock p*, u* is O(eps^2) or smaller
    errs = []
    for eps in (1e-2, 1e-3):
        L = (1.0, 0.3 + eps, 1.0 + 2 * eps)
        R = (1.0 - eps, 0.3, 1.0)
        pe, ue = ex.star(*L, *R, G)
        _, ps, us = ob.h7_riemann([L[0], L[1], 0, 0, L[2]], [R[0], R[1], 0, 0, R[2]], G)
        errs.append(max(abs(ps - pe), abs(us - ue)))
    assert errs[0] < 1e-4 and errs[1] < errs[0] / 50


def test_h7_supersonic_and_mirror_symmetry():
    L = np.array([1.0, 5.0, 0.1, 0.2, 1.0])
    R = np.array([0.8, 4.5, -0.1, -0.2, 0.7])
    out, _, _ = ob.h7_riemann(L, R, G)
    assert out == pytest.approx(L, abs=1e-14)              # everything moves right: face sees L
    for _ in range(50):
        L = np.array([RNG.uniform(0.2, 3), RNG.normal(), RNG.normal(), RNG.normal(), RNG.uniform(0.2, 3)])
        R = np.array([RNG.uniform(0.2, 3), RNG.normal(), RNG.normal(), RNG.normal(), RNG.uniform(0.2, 3)])
        out, ps, us = ob.h7_riemann(L, R, G)
        Lm, Rm = R.copy(), L.copy()
        Lm[1], Rm[1] = -R[1], -L[1]
        om, psm, usm = ob.h7_riemann(Lm, Rm, G)
        assert psm == pytest.approx(ps, rel=1e-13) and usm == pytest.approx(-us, abs=1e-13)
        if abs(us) > 1e-9:
            assert om[[0, 4]] == pytest.approx(out[[0, 4]], rel=1e-12) and om[1] == pytest.approx(-out[1], abs=1e-12)
        # sampled state vs the exact solver's when both waves are shocks
        pe, ue = ex.star(L[0], L[1], L[4], R[0], R[1], R[4], G)
        if pe > max(L[4], R[4]) * 1.0001:
            re_, ue_, pe_ = ex.sample(L[0], L[1], L[4], R[0], R[1], R[4], G, 0.0)
            assert out[[0, 1, 4]] == pytest.approx([re_, ue_, pe_], rel=2e-6, abs=2e-6)


def test_h7_rarefaction_fan_sampling_is_continuous_and_bounded():
    # transonic left rarefaction: sampled state lies between K state and star state
    L = np.array([1.0, 0.9, 0, 0, 1.0])
    R = np.array([0.1, 0.9, 0, 0, 0.05])
    out, ps, us = ob.h7_riemann(L, R, G)
    assert ps < 1.0 and us > 0
    assert ps <= out[4] <= 1.0 and 0.9 <= out[1] <= us
    re_, ue_, pe_ = ex.sample(1.0, 0.9, 1.0, 0.1, 0.9, 0.05, G, 0.0)
    assert out[[0, 1, 4]] == pytest.approx([re_, ue_, pe_], rel=0.2)    # linear-in-fan + two-shock approximation


# ---------------------------------------------------------------- P2 ----------------
def _fv_poly_at(m, pts):
    x, y, z = pts.T
    P2 = lambda s: s * s - 1.0 / 12.0
    return (m[0] + m[1] * x + m[2] * y + m[3] * z + m[4] * P2(x) + m[5] * P2(y) + m[6] * P2(z)
            + m[7] * x * y + m[8] * x * z + m[9] * y * z)


def test_p2_theta_cases_and_bound():
    assert ob.p2_theta([0.5, 0.1, -0.1, 0.05, 0, 0, 0, 0, 0, 0]) == 1.0
    assert ob.p2_theta([0.0, 0.1, 0, 0, 0, 0, 0, 0, 0, 0]) == 0.0
    assert ob.p2_theta([1.0, 0.1, 0, 0, 0.2, 0, 0, 0, 0, 0]) == 0.0
    assert ob.p2_theta([0.5, 0, 0, 0, 0, 0, 0, 0, 0, 0]) == 1.0
    # hand value: m000 = 0.1, B = 0.5*0.4 = 0.2 -> theta = 0.5
    assert ob.p2_theta([0.1, 0.4, 0, 0, 0, 0, 0, 0, 0, 0]) == pytest.approx(0.5)
    pts = RNG.uniform(-0.5, 0.5, size=(4000, 3))
    corners = np.array([[a, b, c] for a in (-.5, .5) for b in (-.5, .5) for c in (-.5, .5)])
    pts = np.vstack([pts, corners])
    for _ in range(200):
        m = RNG.normal(size=10) * RNG.uniform(0, 2)
        m[0] = RNG.uniform(0, 1)
        th = ob.p2_theta(m)
        assert 0.0 <= th <= 1.0
        ms = m.copy()
        ms[1:] *= th
        v = _fv_poly_at(ms, pts)
        assert v.min() >= -1e-12 and v.max() <= 1 + 1e-12


# ---------------------------------------------------------------- P4 -------------------------------
def _cell_poly(a):
    return Poly([a[0] - a[2] / 12.0, a[1], a[2]])


def _brute_remap(deg, a, M, dMl, dMr):
    """independent exact projection with numpy polynomial algebra"""
    Mn = M[1] - dMr + dMl
    pieces = []
    if dMl > 0:
        pieces.append((0, 0.5 - dMl / M[0], 0.5))
    pieces.append((1, -0.5 + max(-dMl, 0) / M[1], 0.5 - max(dMr, 0) / M[1]))
    if dMr < 0:
        pieces.append((2, -0.5, -0.5 - dMr / M[2]))
    basis = [Poly([1.0]), Poly([0.0, 1.0]), Poly([-1.0 / 12.0, 0.0, 1.0])]
    norm = [1.0, 1.0 / 12.0, 1.0 / 180.0]
    out = np.zeros(deg + 1)
    pos = -0.5
    for src, lo, hi in pieces:
        w = (hi - lo) * M[src] / Mn
        # old s as affine function of new s': s = lo + (s' - pos) * (hi - lo) / w
        aff = Poly([lo - pos * (hi - lo) / w, (hi - lo) / w]) if w > 0 else Poly([lo])
        comp = _cell_poly(a[src])(aff)
        for n in range(deg + 1):
            I = (comp * basis[n]).integ()
            out[n] += (I(pos + w) - I(pos)) / norm[n]
        pos += w
    return out


def test_p4_worked_values():
    # donor == 1, own == 0; sigma = 1/2 and 1/4, unit masses
    a = [[1, 0, 0], [0, 0, 0], [0, 0, 0]]
    out, ok = ob.p4_remap(2, a, [1, 1, 1], 0.5, 0.5)
    assert ok and out == pytest.approx([0.5, -1.5, 0.0], abs=1e-13)
    out, _ = ob.p4_remap(2, a, [1, 1, 1], 0.25, 0.25)
    assert out == pytest.approx([0.25, -9.0 / 8.0, 45.0 / 16.0], abs=1e-13)
    b = [[0.3, 0.2, -0.1], [0.6, -0.4, 0.3], [0.1, 0.1, 0.1]]
    out, _ = ob.p4_remap(2, b, [1, 1, 1], 0.0, 0.0)
    assert out == pytest.approx(b[1], abs=1e-14)           # sigma = 0: unchanged
    out, _ = ob.p4_remap(2, b, [1, 1, 1], 1.0, 1.0)
    assert out == pytest.approx(b[0], abs=1e-13)           # sigma = 1: donor's coefficients
    out, _ = ob.p4_remap(2, b, [1, 1, 1], -1.0, -1.0)
    assert out == pytest.approx(b[2], abs=1e-13)           # sigma = -1: right donor's coefficients


def test_p4_closed_form_uniform_flow():
    for _ in range(30):
        s = RNG.uniform(0, 1)
        a0, a1, a2, b0, b1, b2 = RNG.normal(size=6)
        e0 = s * a0 + (1 - s) * b0 + 0.5 * s * (1 - s) * (a1 - b1) + (s ** 3 / 3 - s ** 2 / 2 + s / 6) * (a2 - b2)
        e1 = (6 * s * (s - 1) * (a0 - b0) + (-2 * s ** 3 + 6 * s ** 2 - 3 * s) * a1 + (2 * s ** 3 - 3 * s + 1) * b1
              + (s ** 4 - 4 * s ** 3 + 4 * s ** 2 - s) * a2 + (-s ** 4 + 2 * s ** 2 - s) * b2)
        e2 = (30 * s * (2 * s ** 2 - 3 * s + 1) * (a0 - b0) + 15 * s * (-s ** 3 + 4 * s ** 2 - 4 * s + 1) * a1
              + 15 * s * (s ** 3 - 2 * s + 1) * b1 + (6 * s ** 5 - 30 * s ** 4 + 50 * s ** 3 - 30 * s ** 2 + 5 * s) * a2
              + (-6 * s ** 5 + 10 * s ** 3 - 5 * s + 1) * b2)
        rho_dx = 1.7
        out, _ = ob.p4_remap(2, [[a0, a1, a2], [b0, b1, b2], [9, 9, 9]], [rho_dx] * 3, s * rho_dx, s * rho_dx)
        assert out == pytest.approx([e0, e1, e2], abs=1e-12)


def test_p4_matches_brute_force_projection_all_sign_cases():
    for _ in range(300):
        a = RNG.normal(size=(3, 3))
        M = RNG.uniform(0.5, 2.0, size=3)
        dMl = RNG.uniform(-0.24, 0.24)
        dMr = RNG.uniform(-0.24, 0.24)
        for deg in (0, 1, 2):
            aa = a.copy()
            aa[:, deg + 1:] = 0.0
            out, ok = ob.p4_remap(deg, aa, M, dMl, dMr)
            assert ok
            assert out == pytest.approx(_brute_remap(deg, aa, M, dMl, dMr), abs=1e-11)


def test_p4_quadratic_field_translates_exactly():
    for s in (0.1, 0.37, 0.8, -0.25, -0.6):
        for i in (-3, 0, 2):
            cells = [[(j) ** 2 + 1.0 / 12.0, 2.0 * j, 1.0] for j in (i - 1, i, i + 1)]
            out, _ = ob.p4_remap(2, cells, [1.0, 1.0, 1.0], s, s)
            assert out == pytest.approx([(i - s) ** 2 + 1.0 / 12.0, 2.0 * (i - s), 1.0], abs=1e-12)


def test_p4_mass_conservation_on_a_ring():
    n = 16
    a = RNG.normal(size=(n, 3))
    M = RNG.uniform(0.5, 2.0, size=n)
    dM = RNG.uniform(-0.4, 0.4, size=n)          # dM[j] = mass through the left face of cell j
    tot0 = np.sum(M * a[:, 0])
    tot1 = 0.0
    for j in range(n):
        jm, jp = (j - 1) % n, (j + 1) % n
        out, _ = ob.p4_remap(2, [a[jm], a[j], a[jp]], [M[jm], M[j], M[jp]], dM[j], dM[jp])
        tot1 += (M[j] - dM[jp] + dM[j]) * out[0]
    assert tot1 == pytest.approx(tot0, rel=1e-13)


def test_p4_degenerate_new_mass_leaves_cell_unchanged():
    out, ok = ob.p4_remap(2, [[1, 0, 0], [0.3, 0.2, 0.1], [0, 0, 0]], [1, 1, 1], 0.0, 1.0)
    assert ok == 0 and out == pytest.approx([0.3, 0.2, 0.1])


# ---------------------------------------------------------------- the paper's printed arithmetic ----
def test_paper_printed_arithmetic():
    """tests/golden/paper_arithmetic.txt holds the numbers PAPER.md prints at L149/L118.  They pin reading R18
    (the garbled brick-cost formula) and the record/flop arithmetic DESIGN.md quotes: 64 cells x 16 vars x 4 B,
    2 x 1300 x 32 flops per briquette (L124: 1300-1400 flops per 32-cell half-briquette)."""
    import os
    vals = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_arithmetic.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            vals[line[0]] = float(line[1])
    cost = lambda M: (M + 1) * ((M + 2) ** 2 + (M + 2) * M + M * M)          # R18
    assert cost(40) == vals["brick_updates_M40"] and cost(80) == vals["brick_updates_M80"]
    assert 4 * 4 * 4 * 16 * 4 == vals["briquette_bytes"]
    assert 2 * 1300 * 32 == vals["flops_per_briquette"]
    halo = lambda M: ((M + 2) ** 3 - M ** 3) * 4000 / 1e6       # the paper rounds the 4096-byte record to "4 KB" = 4000 B here
    assert halo(40) == pytest.approx(vals["halo_mbytes_M40"], rel=2e-3)
    assert halo(80) == pytest.approx(vals["halo_mbytes_M80"], rel=2e-3)
    assert cost(40) * vals["flops_per_briquette"] / 1e9 == pytest.approx(vals["gflop_M40"], rel=2e-3)
    assert cost(80) * vals["flops_per_briquette"] / 1e9 == pytest.approx(vals["gflop_M80"], rel=2e-3)
