"""Textbook EXACT Riemann solver for the ideal-gas Euler equations (iterative, Toro ch. 4), written
separately for the tests: it pins the oracle's two-shock solver and the
shock-tube convergence test.  Shares nothing with oracle/ or the CUDA path.
Every function takes an optional `gr`: the adiabatic index of the gas RIGHT of the contact (two-fluid shock tube, NEXT-4;
the contact separates the two gases, so each side's wave uses its own index); default: the same gas on both sides."""
import math

import numpy as np


def _f(p, rk, pk, g):
    ak = 2.0 / ((g + 1.0) * rk)
    bk = (g - 1.0) / (g + 1.0) * pk
    ck = math.sqrt(g * pk / rk)
    if p > pk:
        return (p - pk) * math.sqrt(ak / (p + bk)), math.sqrt(ak / (p + bk)) * (1.0 - 0.5 * (p - pk) / (p + bk))
    return (2.0 * ck / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0),
            1.0 / (rk * ck) * (p / pk) ** (-(g + 1.0) / (2.0 * g)))


def star(rl, ul, pl, rr, ur, pr, g, gr=None):
    gr = g if gr is None else gr
    p = max(1e-12, 0.5 * (pl + pr))
    for _ in range(200):
        fl, dfl = _f(p, rl, pl, g)
        fr, dfr = _f(p, rr, pr, gr)
        pn = max(1e-14, p - (fl + fr + ur - ul) / (dfl + dfr))
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, gr)
    return p, 0.5 * (ul + ur) + 0.5 * (fr - fl)


def sample(rl, ul, pl, rr, ur, pr, g, xi, gr=None):
    """(rho, u, p) of the exact solution at x/t = xi."""
    ps, us = star(rl, ul, pl, rr, ur, pr, g, gr)
    if xi > us and gr is not None:
        g = gr                      # right of the contact: the other gas
    gm = (g - 1.0) / (g + 1.0)
    if xi <= us:
        cl = math.sqrt(g * pl / rl)
        if ps > pl:
            sl = ul - cl * math.sqrt((g + 1.0) / (2.0 * g) * ps / pl + (g - 1.0) / (2.0 * g))
            if xi <= sl:
                return rl, ul, pl
            return rl * (ps / pl + gm) / (gm * ps / pl + 1.0), us, ps
        shl = ul - cl
        csl = cl * (ps / pl) ** ((g - 1.0) / (2.0 * g))
        stl = us - csl
        if xi <= shl:
            return rl, ul, pl
        if xi >= stl:
            return rl * (ps / pl) ** (1.0 / g), us, ps
        c = 2.0 / (g + 1.0) * (cl + 0.5 * (g - 1.0) * (ul - xi))
        return rl * (c / cl) ** (2.0 / (g - 1.0)), 2.0 / (g + 1.0) * (cl + 0.5 * (g - 1.0) * ul + xi), pl * (c / cl) ** (2.0 * g / (g - 1.0))
    cr = math.sqrt(g * pr / rr)
    if ps > pr:
        sr = ur + cr * math.sqrt((g + 1.0) / (2.0 * g) * ps / pr + (g - 1.0) / (2.0 * g))
        if xi >= sr:
            return rr, ur, pr
        return rr * (ps / pr + gm) / (gm * ps / pr + 1.0), us, ps
    shr = ur + cr
    csr = cr * (ps / pr) ** ((g - 1.0) / (2.0 * g))
    strr = us + csr
    if xi >= shr:
        return rr, ur, pr
    if xi <= strr:
        return rr * (ps / pr) ** (1.0 / g), us, ps
    c = 2.0 / (g + 1.0) * (cr - 0.5 * (g - 1.0) * (ur - xi))
    return rr * (c / cr) ** (2.0 / (g - 1.0)), 2.0 / (g + 1.0) * (-cr + 0.5 * (g - 1.0) * ur + xi), pr * (c / cr) ** (2.0 * g / (g - 1.0))


def profile(rl, ul, pl, rr, ur, pr, g, x, x0, t, gr=None):
    return np.array([sample(rl, ul, pl, rr, ur, pr, g, (xx - x0) / t, gr) for xx in x])
