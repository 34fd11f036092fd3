"""ctypes binding of the fp64 CPU oracle (oracle/ppm_oracle.c) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It does not import the CUDA package and the CUDA package does not import it.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

BC_PERIODIC, BC_REFLECT, BC_OPEN = 0, 1, 2
GRAV_NONE, GRAV_CONST_Z, GRAV_RADIAL = 0, 1, 2
NF = 15
FIELD_NAMES = ("rho", "ux", "uy", "uz", "p", "m000", "m100", "m010", "m001",
               "m200", "m020", "m002", "m110", "m101", "m011")

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        fp = C.POINTER(C.c_float)
        ip = C.POINTER(C.c_int)
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, ip, C.c_double, C.c_double, C.c_double, C.c_double,
                                    C.c_int, C.c_int, C.c_double, C.c_double, dp, fp, fp, fp, ip]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_set_state.argtypes = [C.c_void_p, C.POINTER(fp)]
        L.oracle_get_state.argtypes = [C.c_void_p, C.POINTER(dp)]
        L.oracle_raw_field.restype = dp
        L.oracle_raw_field.argtypes = [C.c_void_p, C.c_int]
        L.oracle_sweep.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.oracle_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.oracle_advect.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.oracle_advect_pencil.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, dp, C.POINTER(dp), C.POINTER(dp)]
        L.oracle_set_flatten3d.argtypes = [C.c_void_p, C.c_int]
        L.oracle_flatten3d_update.argtypes = [C.c_void_p]
        L.oracle_flatten3d_field.argtypes = [C.c_void_p]
        L.oracle_flatten3d_field.restype = C.POINTER(C.c_double)
        L.oracle_cfl_dt.argtypes = [C.c_void_p, C.c_double, dp]
        L.oracle_set_sphere.argtypes = [C.c_void_p, C.c_int, C.c_double, dp]
        L.oracle_cell_is_solid.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.oracle_spin_up.argtypes = [C.c_void_p, C.c_double]
        L.oracle_reduce_conserved.argtypes = [C.c_void_p, dp]
        L.oracle_set_two_fluid.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double]
        L.oracle_mix_beta.restype = C.c_double
        L.oracle_mix_beta.argtypes = [C.c_double] * 3
        L.oracle_mix_gamma.restype = C.c_double
        L.oracle_mix_gamma.argtypes = [C.c_double] * 3
        L.oracle_h7_riemann_2f.argtypes = [dp, dp, C.c_double, C.c_double, C.c_double, C.c_double, dp, dp, dp, dp]
        L.oracle_h1_face.restype = C.c_double
        L.oracle_h1_face.argtypes = [C.c_double] * 4
        L.oracle_h2_limit.argtypes = [C.c_double] * 5 + [dp, dp]
        L.oracle_h3_S.restype = C.c_double
        L.oracle_h3_S.argtypes = [dp]
        L.oracle_h3_omega.restype = C.c_double
        L.oracle_h3_omega.argtypes = [C.c_double]
        L.oracle_h4_ftilde.restype = C.c_double
        L.oracle_h4_ftilde.argtypes = [dp, C.c_double, C.c_double, C.c_double]
        L.oracle_h5_Fplus.restype = C.c_double
        L.oracle_h5_Fplus.argtypes = [C.c_double] * 4
        L.oracle_h5_Fminus.restype = C.c_double
        L.oracle_h5_Fminus.argtypes = [C.c_double] * 4
        L.oracle_h6_trace.argtypes = [dp, dp, dp, C.c_double, C.c_double, C.c_double, dp, dp, dp]
        L.oracle_h7_riemann.argtypes = [dp, dp, C.c_double, C.c_double, C.c_double, dp, dp, dp]
        L.oracle_p2_theta.restype = C.c_double
        L.oracle_p2_theta.argtypes = [dp]
        L.oracle_p4_remap.argtypes = [C.c_int, dp, dp, C.c_double, C.c_double, dp]
        L.oracle_sweep_pencil.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                          C.c_double, C.POINTER(dp), C.POINTER(dp), dp, dp, dp, dp, dp,
                                          C.POINTER(dp), C.POINTER(dp), dp]
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _arr(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


# ---- 1-D routine wrappers (used by the pins) -------------------------------------------------
def h1_face(qm1, q0, qp1, qp2):
    return lib().oracle_h1_face(qm1, q0, qp1, qp2)


def h2_limit(qm, qi, qp, fl, fr):
    a, b = C.c_double(), C.c_double()
    lib().oracle_h2_limit(qm, qi, qp, fl, fr, C.byref(a), C.byref(b))
    return a.value, b.value


def h3_S(q5):
    q5 = _arr(q5)
    return lib().oracle_h3_S(_d(q5))


def h3_omega(S):
    return lib().oracle_h3_omega(S)


def h4_ftilde(p5, um, up, ci):
    p5 = _arr(p5)
    return lib().oracle_h4_ftilde(_d(p5), um, up, ci)


def h5_Fplus(ql, qr, qi, s):
    return lib().oracle_h5_Fplus(ql, qr, qi, s)


def h5_Fminus(ql, qr, qi, s):
    return lib().oracle_h5_Fminus(ql, qr, qi, s)


def h6_trace(ql, qr, qi, rho, c, dtdx, src=(0.0, 0.0, 0.0)):
    ql, qr, qi, src = _arr(ql), _arr(qr), _arr(qi), _arr(src)
    WL, WR = np.zeros(5), np.zeros(5)
    lib().oracle_h6_trace(_d(ql), _d(qr), _d(qi), rho, c, dtdx, _d(src), _d(WL), _d(WR))
    return WL, WR


def h7_riemann(L, R, gamma, rho_floor=1e-30, p_floor=1e-30):
    """L, R = (rho, u, v, w, p).  Returns (sampled[5], pstar, ustar)."""
    L, R = _arr(L), _arr(R)
    out = np.zeros(5)
    ps, us = C.c_double(), C.c_double()
    lib().oracle_h7_riemann(_d(L), _d(R), gamma, rho_floor, p_floor, _d(out), C.byref(ps), C.byref(us))
    return out, ps.value, us.value


def h7_riemann_2f(L, R, gamL, gamR, rho_floor=1e-30, p_floor=1e-30):
    """NEXT-4: H7 with one adiabatic index per side.  Returns (sampled[5], gamma of the sampled side, pstar, ustar)."""
    L, R = _arr(L), _arr(R)
    out = np.zeros(5)
    gh, ps, us = C.c_double(), C.c_double(), C.c_double()
    lib().oracle_h7_riemann_2f(_d(L), _d(R), gamL, gamR, rho_floor, p_floor, _d(out), C.byref(gh), C.byref(ps), C.byref(us))
    return out, gh.value, ps.value, us.value


def mix_beta(f, gamma1, gamma2):
    return lib().oracle_mix_beta(f, gamma1, gamma2)


def mix_gamma(f, gamma1, gamma2):
    return lib().oracle_mix_gamma(f, gamma1, gamma2)


def p2_theta(m10):
    m10 = _arr(m10)
    return lib().oracle_p2_theta(_d(m10))


def p4_remap(deg, a3x3, M3, dMl, dMr):
    a = _arr(a3x3).reshape(3, 3)
    M = _arr(M3)
    out = np.zeros(3)
    ok = lib().oracle_p4_remap(deg, _d(a), _d(M), dMl, dMr, _d(out))
    return out[:deg + 1].copy(), ok


def sweep_pencil(d, dx, dt, gamma, q5, m10, rho0c=None, p0c=None, gd=None, rho0f=None, p0f=None,
                 rho_floor=1e-30, p_floor=1e-30, ft_ext=None):
    """q5: (5, n+8) = rho', u_normal, v, w, p' with ghosts; m10: (10, n+8).  Returns (5,n), (10,n).
    ft_ext: (n+8,) un-spread flattening coefficients that replace the 1-D detector (3-D flattening mode)."""
    q5, m10 = _arr(q5), _arr(m10)
    nt = q5.shape[1]
    n = nt - 8
    z = np.zeros(nt + 1)
    rho0c = _arr(rho0c) if rho0c is not None else z[:nt].copy()
    p0c = _arr(p0c) if p0c is not None else z[:nt].copy()
    gd = _arr(gd) if gd is not None else z[:nt].copy()
    rho0f = _arr(rho0f) if rho0f is not None else z.copy()
    p0f = _arr(p0f) if p0f is not None else z.copy()
    qo, mo = np.zeros((5, n)), np.zeros((10, n))
    dp = C.POINTER(C.c_double)
    qi = (dp * 5)(*[_d(q5[k]) for k in range(5)])
    mi = (dp * 10)(*[_d(m10[k]) for k in range(10)])
    qop = (dp * 5)(*[_d(qo[k]) for k in range(5)])
    mop = (dp * 10)(*[_d(mo[k]) for k in range(10)])
    lib().oracle_sweep_pencil(n, d, dx, dt, gamma, rho_floor, p_floor, qi, mi, _d(rho0c), _d(p0c), _d(gd),
                              _d(rho0f), _d(p0f), qop, mop, _d(_arr(ft_ext)) if ft_ext is not None else None)
    return qo, mo


def advect_pencil(d, dx, dt, u, m10):
    """u: (n+8,) normal velocity with ghosts; m10: (10, n+8).  Returns (10, n)."""
    u, m10 = _arr(u), _arr(m10)
    n = u.size - 8
    mo = np.zeros((10, n))
    dp = C.POINTER(C.c_double)
    mi = (dp * 10)(*[_d(m10[k]) for k in range(10)])
    mop = (dp * 10)(*[_d(mo[k]) for k in range(10)])
    lib().oracle_advect_pencil(n, d, dx, dt, _d(u), mi, mop)
    return mo


def num_threads():
    return lib().oracle_num_threads()


# ---- 3-D driver --------------------------------------------------------------------------------
class Oracle:
    """fp64 oracle on a full grid or on a window (org != 0, OPEN sides) of a larger grid."""

    def __init__(self, nx, ny, nz, dx, gamma, bc, grav=None, org=(0, 0, 0), rho_floor=1e-30, p_floor=1e-30):
        self.shape = (nz, ny, nx)
        self.n = (nx, ny, nz)
        kind, n, s0, ds, center = GRAV_NONE, 0, 0.0, 1.0, (0.0, 0.0, 0.0)
        g = r0 = p0 = None
        if grav is not None and grav["kind"] != GRAV_NONE:
            kind, s0, ds = int(grav["kind"]), float(grav["s0"]), float(grav["ds"])
            center = tuple(grav.get("center", (0.0, 0.0, 0.0)))
            g = np.ascontiguousarray(grav["g"], dtype=np.float32)
            r0 = np.ascontiguousarray(grav["rho0"], dtype=np.float32)
            p0 = np.ascontiguousarray(grav["p0"], dtype=np.float32)
            n = g.size
        self._keep = (g, r0, p0)
        fp = C.POINTER(C.c_float)
        fptr = lambda a: a.ctypes.data_as(fp) if a is not None else None
        org_a = (C.c_int * 3)(*[int(v) for v in org])
        bc_a = (C.c_int * 6)(*[int(v) for v in bc])
        cen = (C.c_double * 3)(*[float(v) for v in center])
        self._h = lib().oracle_create(nx, ny, nz, org_a, dx, gamma, rho_floor, p_floor, kind, n, s0, ds,
                                      cen, fptr(g), fptr(r0), fptr(p0), bc_a)
        if not self._h:
            raise ValueError("oracle_create rejected the parameters")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, fields):
        """fields: sequence of 15 float32 arrays [nz][ny][nx] (full rho, u, p, moments)."""
        arrs = [np.ascontiguousarray(f, dtype=np.float32) for f in fields]
        assert len(arrs) == NF and all(a.shape == self.shape for a in arrs)
        fp = C.POINTER(C.c_float)
        ptrs = (fp * NF)(*[a.ctypes.data_as(fp) for a in arrs])
        rc = lib().oracle_set_state(self._h, ptrs)
        assert rc == 0

    def get_state(self):
        out = np.zeros((NF,) + self.shape, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        ptrs = (dp * NF)(*[_d(out[f]) for f in range(NF)])
        rc = lib().oracle_get_state(self._h, ptrs)
        assert rc == 0
        return out

    def raw_field(self, f):
        p = lib().oracle_raw_field(self._h, f)
        return np.ctypeslib.as_array(p, shape=self.shape)

    def set_flatten3d(self, on=True):
        """NEXT-1: fully 3-D shock detector instead of the per-sweep 1-D one"""
        rc = lib().oracle_set_flatten3d(self._h, int(bool(on)))
        if rc:
            raise ValueError("oracle_set_flatten3d rc=%d" % rc)

    def flatten3d_field(self, update=True):
        """F~ [nz][ny][nx] evaluated on the current state"""
        if update:
            lib().oracle_flatten3d_update(self._h)
        ptr = lib().oracle_flatten3d_field(self._h)
        return np.ctypeslib.as_array(ptr, shape=self.shape).copy()

    def set_sphere(self, radius, center):
        """NEXT-3: confining sphere; radius <= 0 switches it off"""
        cen = (C.c_double * 3)(*[float(v) for v in center])
        rc = lib().oracle_set_sphere(self._h, int(radius > 0), float(radius), cen)
        if rc:
            raise ValueError("oracle_set_sphere rc=%d" % rc)

    def set_two_fluid(self, gamma1, gamma2):
        """NEXT-4: two-fluid EOS (reading R25): gamma1 = the tracked fluid (FV), gamma2 =
        the rest.  gamma1 = None switches it off."""
        rc = lib().oracle_set_two_fluid(self._h, int(gamma1 is not None), float(gamma1 or 0.0), float(gamma2 or 0.0))
        if rc:
            raise ValueError("oracle_set_two_fluid rc=%d" % rc)

    def solid_mask(self):
        """bool [nz][ny][nx]: cells whose centre lies outside the confining sphere"""
        nz, ny, nx = self.shape
        L = lib()
        return np.array([[[bool(L.oracle_cell_is_solid(self._h, i, j, k)) for i in range(nx)] for j in range(ny)]
                         for k in range(nz)])

    def spin_up(self, domega):
        """NEXT-3: one increment of the solid-body rotation ramp about z"""
        rc = lib().oracle_spin_up(self._h, float(domega))
        assert rc == 0

    def sweep(self, d, dt):
        rc = lib().oracle_sweep(self._h, d, dt)
        assert rc == 0

    def advect(self, dt, order=0):
        """NEXT-2: PPB-only step (FV advected by the stored velocity field, hydro state held fixed)"""
        rc = lib().oracle_advect(self._h, dt, order)
        if rc:
            raise ValueError("oracle_advect rc=%d" % rc)

    def step(self, dt, order=0):
        rc = lib().oracle_step(self._h, dt, order)
        if rc != 0:
            raise ValueError("oracle_step rc=%d" % rc)

    def cfl_dt(self, cfl):
        v = C.c_double()
        lib().oracle_cfl_dt(self._h, cfl, C.byref(v))
        return v.value

    def reduce_conserved(self):
        out = np.zeros(6)
        lib().oracle_reduce_conserved(self._h, _d(out))
        return out
