"""TEST-ONLY comparator for reading R8': a plain numpy 1-D direct-Eulerian PPM hydro sweep
(SURVEY.md 8(c) H0-H9 without gravity and without PPB) whose characteristic tracing can be switched between

  "r8p"  : the oracle's switch-free tracing (every family takes its amplitude over max(+-sigma^k, 0); a wave that
           leaves the face has the zero-width domain, i.e. the edge value), and
  "cw84" : the hard-switched tracing of Colella & Woodward 1984 (PAPER.md L87 -> ref. [30], L189): the terms of a
           family are present only if its characteristic moves toward the face (SURVEY.md 8(c) H6 as first written).

It exists to measure how far R8' moves the SOLUTION from the textbook scheme (tests/test_oracle_r8prime.py).  It is
not an oracle, not a pin, and nothing under oracle/ or the CUDA package uses it.
"""
import numpy as np

TINY = 1e-30


def _med(a, b, c):
    return np.maximum(np.minimum(a, b), np.minimum(np.maximum(a, b), c))


def _clamp01(x):
    return np.minimum(1.0, np.maximum(0.0, x))


def _ghosts(q, ng, bc, odd=False):
    if bc == "periodic":
        return np.concatenate([q[-ng:], q, q[:ng]])
    s = -1.0 if odd else 1.0
    return np.concatenate([s * q[ng - 1::-1], q, s * q[:-ng - 1:-1]])


def _Fp(ql, qr, qi, s):
    dq, q6 = qr - ql, 6.0 * (qi - 0.5 * (ql + qr))
    return qr - 0.5 * s * (dq - (1.0 - 2.0 * s / 3.0) * q6)


def _Fm(ql, qr, qi, s):
    dq, q6 = qr - ql, 6.0 * (qi - 0.5 * (ql + qr))
    return ql + 0.5 * s * (dq + (1.0 - 2.0 * s / 3.0) * q6)


def riemann_two_shock(L, R, gamma, floor=1e-30):
    """H7, vectorised: L, R = dicts rho,u,p (arrays).  Returns sampled rho, u, p at x/t = 0 and the upwind mask."""
    rl, ul, pl, rr, ur, pr = L["rho"], L["u"], L["p"], R["rho"], R["u"], R["p"]
    CL, CR = np.sqrt(gamma * pl * rl), np.sqrt(gamma * pr * rr)
    gp, gm = 0.5 * (gamma + 1.0), 0.5 * (gamma - 1.0)
    ps = np.maximum(floor, (CR * pl + CL * pr + CL * CR * (ul - ur)) / (CL + CR))
    for _ in range(5):
        WL, WR = np.sqrt(rl * (gp * ps + gm * pl)), np.sqrt(rr * (gp * ps + gm * pr))
        usl, usr = ul - (ps - pl) / WL, ur + (ps - pr) / WR
        ZL, ZR = 2.0 * WL ** 3 / (WL * WL + CL * CL), 2.0 * WR ** 3 / (WR * WR + CR * CR)
        ps = np.maximum(floor, ps - ZL * ZR * (usr - usl) / (ZL + ZR))
    WL, WR = np.sqrt(rl * (gp * ps + gm * pl)), np.sqrt(rr * (gp * ps + gm * pr))
    us = (WL * ul + WR * ur + pl - pr) / (WL + WR)
    left = us >= 0.0
    s = np.where(left, 1.0, -1.0)
    rK, uK, pK, WK = np.where(left, rl, rr), np.where(left, ul, ur), np.where(left, pl, pr), np.where(left, WL, WR)
    rs = np.maximum(1.0 / (1.0 / rK - (ps - pK) / (WK * WK)), floor)
    cK, cs = np.sqrt(gamma * pK / rK), np.sqrt(gamma * ps / rs)
    uKh, ush = s * uK, s * us
    shock = ps > pK
    head = np.where(shock, uKh - WK / rK, uKh - cK)
    tail = np.where(shock, head, ush - cs)
    with np.errstate(divide="ignore", invalid="ignore"):
        th = np.where(head >= 0.0, 0.0, np.where(tail <= 0.0, 1.0, -head / (tail - head)))
    return (1 - th) * rK + th * rs, (1 - th) * uK + th * us, (1 - th) * pK + th * ps, left


def sweep(rho, u, p, dt, dx, gamma, bc="periodic", tracing="r8p"):
    """one 1-D hydro sweep (v = w = 0); returns new (rho, u, p)"""
    ng = 4
    n = rho.size
    q = [_ghosts(rho, ng, bc), _ghosts(u, ng, bc, odd=True), _ghosts(p, ng, bc)]
    nt = n + 2 * ng
    r, uu, pp = q
    c = np.sqrt(gamma * pp / r)
    dtdx = dt / dx
    # H1 faces f = 2 .. nt-2 (between cells f-1 and f)
    qu = [np.full(nt + 1, np.nan) for _ in q]
    for k, a in enumerate(q):
        qu[k][2:nt - 1] = (7.0 / 12.0) * (a[1:nt - 2] + a[2:nt - 1]) - (1.0 / 12.0) * (a[0:nt - 3] + a[3:nt])
    # H4
    ft = np.zeros(nt)
    j = np.arange(2, nt - 2)
    d1, d2 = pp[j + 1] - pp[j - 1], pp[j + 2] - pp[j - 2]
    steep = _clamp01(10.0 * (np.abs(d1) / np.maximum(np.abs(d2), TINY) - 0.75))
    jump = _clamp01(3.0 * np.abs(d1) / np.minimum(pp[j + 1], pp[j - 1]) - 1.0)
    conv = _clamp01((uu[j - 1] - uu[j + 1]) / (0.05 * c[j]))
    ft[j] = steep * jump * conv
    fl = np.zeros(nt)
    fl[3:nt - 3] = np.maximum(ft[2:nt - 4], np.maximum(ft[3:nt - 3], ft[4:nt - 2]))
    # H2, H3 for cells 3 .. nt-4
    j = np.arange(3, nt - 3)
    ql, qr = [], []
    for k, a in enumerate(q):
        fL, fR = qu[k][j], qu[k][j + 1]
        Lm, Rm = _med(a[j - 1], fL, a[j]), _med(a[j], fR, a[j + 1])
        ext = (Rm - a[j]) * (a[j] - Lm) <= 0.0
        D, q6 = Rm - Lm, 6.0 * (a[j] - 0.5 * (Lm + Rm))
        L2 = np.where(D * q6 > D * D, 3.0 * a[j] - 2.0 * Rm, Lm)
        R2 = np.where((D * q6 < -D * D) & ~(D * q6 > D * D), 3.0 * a[j] - 2.0 * Lm, Rm)
        Lm, Rm = np.where(ext, a[j], L2), np.where(ext, a[j], R2)
        d2m, d20, d2p = a[j] - 2 * a[j - 1] + a[j - 2], a[j + 1] - 2 * a[j] + a[j - 1], a[j + 2] - 2 * a[j + 1] + a[j]
        S = np.abs(d2p - d2m) / (np.abs(d2m) + 2.0 * np.abs(d20) + np.abs(d2p) + TINY)
        om = _clamp01((S - 0.1) / 0.2)
        L, R = (1 - om) * fL + om * Lm, (1 - om) * fR + om * Rm
        ql.append(fl[j] * a[j] + (1 - fl[j]) * L)
        qr.append(fl[j] * a[j] + (1 - fl[j]) * R)
    # H5, H6
    qi = [a[j] for a in q]
    ri, ci, ui = r[j], c[j], uu[j]
    s_m, s_0, s_p = (ui - ci) * dtdx, ui * dtdx, (ui + ci) * dtdx
    c2 = ci * ci
    FP = lambda k, s: _Fp(ql[k], qr[k], qi[k], s)
    FM = lambda k, s: _Fm(ql[k], qr[k], qi[k], s)
    # left of face j+1/2
    sp = np.maximum(s_p, 0.0)
    rt, ut, pt = FP(0, sp), FP(1, sp), FP(2, sp)
    if tracing == "r8p":
        smk, s0k = np.maximum(s_m, 0.0), np.maximum(s_0, 0.0)
        on_m = on_0 = 1.0
    else:
        smk, s0k = s_m, s_0
        on_m, on_0 = (s_m > 0.0) * 1.0, (s_0 > 0.0) * 1.0
    am = on_m * ((pt - FP(2, smk)) - ri * ci * (ut - FP(1, smk))) / (2.0 * c2)
    a0 = on_0 * ((rt - FP(0, s0k)) - (pt - FP(2, s0k)) / c2)
    WL = [rt - am - a0, ut + (ci / ri) * am, pt - c2 * am]
    # right of face j-1/2
    sm = np.maximum(-s_m, 0.0)
    rt, ut, pt = FM(0, sm), FM(1, sm), FM(2, sm)
    if tracing == "r8p":
        spk, s0k = np.maximum(-s_p, 0.0), np.maximum(-s_0, 0.0)
        on_p = on_0 = 1.0
    else:
        spk, s0k = -s_p, -s_0
        on_p, on_0 = (s_p < 0.0) * 1.0, (s_0 < 0.0) * 1.0
    ap = on_p * ((pt - FM(2, spk)) + ri * ci * (ut - FM(1, spk))) / (2.0 * c2)
    a0 = on_0 * ((rt - FM(0, s0k)) - (pt - FM(2, s0k)) / c2)
    WR = [rt - ap - a0, ut - (ci / ri) * ap, pt - c2 * ap]
    # H7, H8 at faces f = 4 .. nt-4: left state from cell f-1 (index f-1-3 in j), right state from cell f (index f-3)
    nf = n + 1
    L = dict(rho=WL[0][0:nf], u=WL[1][0:nf], p=WL[2][0:nf])
    R = dict(rho=WR[0][1:nf + 1], u=WR[1][1:nf + 1], p=WR[2][1:nf + 1])
    rh, uh, ph, _ = riemann_two_shock(L, R, gamma)
    Fm = rh * uh
    Fn = Fm * uh + ph
    FE = uh * (gamma / (gamma - 1.0) * ph + 0.5 * rh * uh * uh)
    # H9
    E0 = p / (gamma - 1.0) + 0.5 * rho * u * u
    r1 = rho - dtdx * (Fm[1:] - Fm[:-1])
    m1 = rho * u - dtdx * (Fn[1:] - Fn[:-1])
    E1 = E0 - dtdx * (FE[1:] - FE[:-1])
    u1 = m1 / r1
    return r1, u1, (gamma - 1.0) * (E1 - 0.5 * r1 * u1 * u1)


def run(rho, u, p, gamma, t_end, cfl, bc="periodic", tracing="r8p", dts=None):
    """march to t_end with dt = cfl dx / max(|u| + c), or with the given list of dt; returns (rho, u, p, dts used)"""
    n = rho.size
    dx = 1.0 / n
    t, used = 0.0, []
    k = 0
    while t < t_end - 1e-14:
        if dts is not None:
            dt = dts[k]
        else:
            dt = min(cfl * dx / np.max(np.abs(u) + np.sqrt(gamma * p / rho)), t_end - t)
        rho, u, p = sweep(rho, u, p, dt, dx, gamma, bc, tracing)
        used.append(dt)
        t += dt
        k += 1
    return rho, u, p, used
