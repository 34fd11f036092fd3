"""Error norms used by the GPU-vs-oracle parity tests.

per-variable max relative error = max_cells |gpu - oracle| / max_cells |oracle|, rho and p on the FULL values.
The ten FV coefficients share one scale, max |m000|: they describe ONE variable (the sub-cell polynomial of
FV), and a coefficient such as m110 that is ~0 by symmetry has no scale of its own — rounding the fp32
STATE alone (fp64 arithmetic) already moves it by 1e-4 of its own maximum within five steps
(tests/test_oracle_invariants.py::test_fp32_state_storage_sets_the_parity_floor; reading R20a).
A velocity component keeps its own scale, floored at 1e-3 of the largest component (degenerate symmetry).
"""
import numpy as np

VARS = ("rho", "u", "p", "FV")


def groups(o):
    """scale per field index"""
    s = np.zeros(15)
    s[0] = np.abs(o[0]).max()
    umax = max(np.abs(o[1:4]).max(), 1e-300)
    for f in (1, 2, 3):
        s[f] = max(np.abs(o[f]).max(), 1e-3 * umax)
    s[4] = np.abs(o[4]).max()
    s[5:] = max(np.abs(o[5]).max(), 1e-300)
    return s


def max_rel(g, o, scale=None):
    """dict var -> max relative error (R20/R20a).  `scale` (15 numbers) overrides the per-field maxima, e.g.
    the maxima over ALL windows of a windowed check (a window inside a quiescent region has no scale)."""
    s = groups(o) if scale is None else scale
    e = np.array([np.abs(g[f] - o[f]).max() / s[f] for f in range(15)])
    return {"rho": e[0], "u": e[1:4].max(), "p": e[4], "FV": e[5:].max()}


def pert_rel(gp, op):
    """The perturbation fields themselves: gp, op = (rho', p') as the GPU stores them
    (ppm_get_state with PPM_OPT_STATE_FORM = 1) and as the oracle stores them (oracle_raw_field 0, 4).
    max |gpu - oracle| / max |oracle| per field — in the low-Mach configs rho', p' are 1e-3 .. 1e-6 of the base state, so
    this norm is that much stricter than the full-value norm of R20; a field the oracle leaves at round-off level
    (max |q'| below 1e-12 of the base scale `floor`) has no scale and reports 0."""
    out = {}
    for name, g, o in (("rho'", gp[0], op[0]), ("p'", gp[1], op[1])):
        sc = np.abs(o).max()
        out[name] = float(np.abs(g - o).max() / sc) if sc > 0 else 0.0
        out[name + " scale"] = float(sc)
    return out


def abs_err(g, o):
    return np.array([np.abs(g[f] - o[f]).max() for f in range(15)])


def merge_scales(list_of_o):
    """per-field scales over several oracle windows"""
    mx = np.max([[np.abs(o[f]).max() for f in range(15)] for o in list_of_o], axis=0)
    fake = [np.array([mx[f]]) for f in range(15)]
    return groups(fake)


def l1_rel(g, o):
    """dict var -> sum |gpu - oracle| / sum |oracle| (the shock-config norm)"""
    d = lambda sl: np.abs(g[sl] - o[sl]).sum() / max(np.abs(o[sl]).sum(), 1e-300)
    return {"rho": d(slice(0, 1)), "u": d(slice(1, 4)), "p": d(slice(4, 5)), "FV": d(slice(5, 15))}


def conserved_rel(cg, co, o_full, dx, gamma):
    """|gpu - oracle| of the six totals relative to sum |summand| (R20)."""
    rho, u, v, w, p, m0 = o_full[0], o_full[1], o_full[2], o_full[3], o_full[4], o_full[5]
    dv = dx ** 3
    scale = np.array([np.abs(rho).sum(), np.abs(rho * u).sum(), np.abs(rho * v).sum(), np.abs(rho * w).sum(),
                      np.abs(p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w)).sum(), np.abs(rho * m0).sum()]) * dv
    return np.abs(np.asarray(cg) - np.asarray(co)) / np.maximum(scale, 1e-300)
