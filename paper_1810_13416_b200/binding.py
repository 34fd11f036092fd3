"""Thin ctypes binding of libppm_b200.so (include/ppm.h).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels.  torch supplies device memory and the stream, nothing else.

Fails loudly (ImportError / RuntimeError) when the library is missing or a call fails; there is no
CPU fallback and this module never imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
# PPM_B200_LIB: load another build of the same library (e.g. one compiled with different tuning knobs)
LIB_PATH = os.environ.get("PPM_B200_LIB") or os.path.join(HERE, "libppm_b200.so")

PPM_OK, PPM_EINVAL, PPM_ENOMEM, PPM_ECUDA, PPM_ESTATE = 0, 1, 2, 3, 4
BC_PERIODIC, BC_REFLECT = 0, 1
GRAV_NONE, GRAV_CONST_Z, GRAV_RADIAL = 0, 1, 2
NF = 15
EXPORTS = ("ppm_create", "ppm_set_state", "ppm_get_state", "ppm_step", "ppm_sweep", "ppm_advect", "ppm_cfl_dt",
           "ppm_reduce_conserved", "ppm_sync", "ppm_set_chunk", "ppm_set_option", "ppm_axis_path", "ppm_launch_count",
           "ppm_state_floats", "ppm_plan_tail_chunk", "ppm_destroy", "ppm_last_error")
OPT_IO_PATH, OPT_FLATTEN3D, OPT_CFL_FUSED = 2, 3, 4


class ppm_gravity(C.Structure):
    _fields_ = [("kind", C.c_int), ("n", C.c_int), ("s0", C.c_double), ("ds", C.c_double),
                ("center", C.c_double * 3), ("g", C.POINTER(C.c_float)), ("rho0", C.POINTER(C.c_float)),
                ("p0", C.POINTER(C.c_float))]


class ppm_params(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("gamma", C.c_double), ("rho_floor", C.c_double), ("p_floor", C.c_double),
                ("grav", ppm_gravity), ("bc", C.c_int * 6), ("stream", C.c_void_p)]


_lib = None


def lib():
    """Load the in-tree library; raise if it is not built (python -m paper_1810_13416_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libppm_b200.so is not built: run `python -m paper_1810_13416_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        fpp = C.POINTER(C.POINTER(C.c_float))
        L.ppm_state_floats.argtypes = [C.c_int, C.c_int, C.c_int]
        L.ppm_state_floats.restype = C.c_size_t
        L.ppm_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(ppm_params), C.c_void_p, C.c_void_p]
        L.ppm_set_state.argtypes = [C.c_void_p, fpp, C.c_int, C.c_int, C.c_int]
        L.ppm_get_state.argtypes = [C.c_void_p, fpp, C.c_int, C.c_int, C.c_int]
        L.ppm_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.ppm_sweep.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.ppm_advect.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.ppm_cfl_dt.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.ppm_reduce_conserved.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.ppm_sync.argtypes = [C.c_void_p]
        L.ppm_set_chunk.argtypes = [C.c_void_p, C.c_int]
        L.ppm_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.ppm_axis_path.argtypes = [C.c_void_p, C.c_int]
        L.ppm_plan_tail_chunk.argtypes = [C.c_int, C.c_int, C.c_int]
        L.ppm_launch_count.argtypes = [C.c_void_p]
        L.ppm_launch_count.restype = C.c_longlong
        L.ppm_destroy.argtypes = [C.c_void_p]
        L.ppm_destroy.restype = None
        L.ppm_last_error.argtypes = [C.c_void_p]
        L.ppm_last_error.restype = C.c_char_p
        _lib = L
    return _lib


class PPMError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("ppm error %d: %s" % (code, msg))
        self.code = code


def make_params(nx, ny, nz, dx, gamma, bc, grav=None, rho_floor=1e-10, p_floor=1e-10, stream=0):
    """Returns (ppm_params, keepalive) — keepalive holds the numpy table arrays the struct points to."""
    p = ppm_params()
    p.struct_size = C.sizeof(ppm_params)
    p.nx, p.ny, p.nz = int(nx), int(ny), int(nz)
    p.dx, p.gamma, p.rho_floor, p.p_floor = float(dx), float(gamma), float(rho_floor), float(p_floor)
    keep = []
    if grav is not None and int(grav["kind"]) != GRAV_NONE:
        fp = C.POINTER(C.c_float)
        arrs = [np.ascontiguousarray(grav[k], dtype=np.float32) for k in ("g", "rho0", "p0")]
        keep = arrs
        p.grav.kind, p.grav.n = int(grav["kind"]), int(arrs[0].size)
        p.grav.s0, p.grav.ds = float(grav["s0"]), float(grav["ds"])
        for d in range(3):
            p.grav.center[d] = float(grav.get("center", (0.0, 0.0, 0.0))[d])
        p.grav.g, p.grav.rho0, p.grav.p0 = (a.ctypes.data_as(fp) for a in arrs)
    else:
        p.grav.kind, p.grav.n, p.grav.s0, p.grav.ds = GRAV_NONE, 0, 0.0, 1.0
    for k in range(6):
        p.bc[k] = int(bc[k])
    p.stream = C.c_void_p(int(stream))
    return p, keep


class PPM:
    """One context = one grid on one GPU.  Owns the two borrowed torch buffers (state + scratch)."""

    def __init__(self, nx, ny, nz, dx, gamma, bc, grav=None, rho_floor=1e-10, p_floor=1e-10, device="cuda:0",
                 stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1810_13416_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        self.n = (int(nx), int(ny), int(nz))
        self.ncell = int(nx) * int(ny) * int(nz)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        nfl = int(lib().ppm_state_floats(int(nx), int(ny), int(nz)))
        with torch.cuda.device(self.device):
            self.buf_a = torch.empty(nfl, dtype=torch.float32, device=self.device)
            self.buf_b = torch.empty(nfl, dtype=torch.float32, device=self.device)
        prm, keep = make_params(nx, ny, nz, dx, gamma, bc, grav, rho_floor, p_floor, self.stream.cuda_stream)
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = lib().ppm_create(C.byref(self._h), C.byref(prm), C.c_void_p(self.buf_a.data_ptr()),
                                  C.c_void_p(self.buf_b.data_ptr()))
        if rc != PPM_OK:
            raise PPMError(rc, lib().ppm_last_error(None).decode())

    @classmethod
    def from_workload(cls, w, device="cuda:0", stream=None):
        return cls(w.n, w.n, w.n, w.dx, w.gamma, w.bc, w.grav, w.rho_floor, w.p_floor, device, stream)

    def _check(self, rc):
        if rc != PPM_OK:
            raise PPMError(rc, lib().ppm_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().ppm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- marshalling helpers ----
    def _ptrs(self, t):
        """t: torch tensor [15, nzs, ny, nx] float32 contiguous (device or host) -> float*[15]"""
        assert t.dtype == torch.float32 and t.is_contiguous() and t.shape[0] == NF
        fp = C.POINTER(C.c_float)
        stride = t.stride(0) * 4
        base = t.data_ptr()
        return (fp * NF)(*[C.cast(C.c_void_p(base + f * stride), fp) for f in range(NF)])

    def set_state(self, fields, z0=0):
        """fields: [15, nzs, ny, nx] float32, torch (cuda or cpu, pinned or not) or numpy."""
        if isinstance(fields, np.ndarray):
            fields = torch.from_numpy(np.ascontiguousarray(fields, dtype=np.float32))
        nzs = fields.shape[1]
        assert tuple(fields.shape[2:]) == (self.n[1], self.n[0])
        self._check(lib().ppm_set_state(self._h, self._ptrs(fields), int(z0), int(nzs), int(fields.is_cuda)))
        if not fields.is_cuda:
            self.stream.synchronize()      # the host source must stay valid until the copy is done

    def get_state(self, z0=0, nzs=None, out=None, device=None):
        nzs = self.n[2] - z0 if nzs is None else nzs
        if out is None:
            out = torch.empty((NF, nzs, self.n[1], self.n[0]), dtype=torch.float32,
                              device=device if device is not None else self.device)
        self._check(lib().ppm_get_state(self._h, self._ptrs(out), int(z0), int(nzs), int(out.is_cuda)))
        return out

    def step(self, dt, order=0):
        self._check(lib().ppm_step(self._h, float(dt), int(order)))

    def advect(self, dt, order=0):
        """PPB-only step: FV advected by the stored velocity field, hydro state held fixed (NEXT-2)"""
        self._check(lib().ppm_advect(self._h, float(dt), int(order)))

    def sweep(self, dt, axis):
        self._check(lib().ppm_sweep(self._h, float(dt), int(axis)))

    def cfl_dt(self, cfl):
        v = C.c_double()
        self._check(lib().ppm_cfl_dt(self._h, float(cfl), C.byref(v)))
        return v.value

    def reduce_conserved(self):
        out = (C.c_double * 6)()
        self._check(lib().ppm_reduce_conserved(self._h, out))
        return np.array(list(out))

    def sync(self):
        self._check(lib().ppm_sync(self._h))

    def set_chunk(self, chunk):
        self._check(lib().ppm_set_chunk(self._h, int(chunk)))

    def set_option(self, option, value):
        self._check(lib().ppm_set_option(self._h, int(option), int(value)))

    def axis_path(self, axis):
        return int(lib().ppm_axis_path(self._h, int(axis)))

    def launch_count(self):
        return int(lib().ppm_launch_count(self._h))
