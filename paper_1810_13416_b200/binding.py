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
STATIC_RED_BLOCKS = 1024      # PPM_STATIC_RED_BLOCKS: first-pass blocks the static scratch array of ppm_reduce_conserved_static holds
BC_PERIODIC, BC_REFLECT, BC_HALO = 0, 1, 2
GRAV_NONE, GRAV_CONST_Z, GRAV_RADIAL = 0, 1, 2
NF = 15
EXPORTS = ("ppm_create", "ppm_set_state", "ppm_get_state", "ppm_step", "ppm_sweep", "ppm_advect", "ppm_cfl_dt",
           "ppm_reduce_conserved", "ppm_reduce_conserved_static", "ppm_sync", "ppm_set_chunk", "ppm_set_option", "ppm_axis_path", "ppm_launch_count",
           "ppm_state_floats", "ppm_plan_tail_chunk", "ppm_measure_fp32_peak", "ppm_set_sphere", "ppm_spin_up", "ppm_set_two_fluid", "ppm_halo_floats", "ppm_pack_halo", "ppm_set_halo",
           "ppm_set_origin", "ppm_sweep_cfl", "ppm_destroy",
           "ppm_last_error")
OPT_IO_PATH, OPT_FLATTEN3D, OPT_CFL_FUSED, OPT_STATE_FORM, OPT_FV_SHORTCUT = 2, 3, 4, 5, 6


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
        L.ppm_reduce_conserved_static.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.ppm_sync.argtypes = [C.c_void_p]
        L.ppm_set_chunk.argtypes = [C.c_void_p, C.c_int]
        L.ppm_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.ppm_axis_path.argtypes = [C.c_void_p, C.c_int]
        L.ppm_plan_tail_chunk.argtypes = [C.c_int, C.c_int, C.c_int]
        L.ppm_launch_count.argtypes = [C.c_void_p]
        L.ppm_launch_count.restype = C.c_longlong
        L.ppm_measure_fp32_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.ppm_set_sphere.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.ppm_spin_up.argtypes = [C.c_void_p, C.c_double]
        L.ppm_set_two_fluid.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.ppm_halo_floats.restype = C.c_size_t
        L.ppm_halo_floats.argtypes = [C.c_int] * 4
        L.ppm_pack_halo.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.ppm_set_halo.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.ppm_set_origin.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
        L.ppm_sweep_cfl.argtypes = [C.c_void_p, C.c_double, C.c_int]
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
        """t: torch tensor [15, nzs, ny, nx] float32 (device or host), every field a dense [nzs][ny][nx] block -> float*[15]"""
        assert t.dtype == torch.float32 and t.shape[0] == NF and t[0].is_contiguous()
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

    def step_host_pipelined(self, host_ins, host_outs, dt, orders, slab=32, step=None, wait=True):
        """End-to-end helper for host-resident grids (argument marshalling and stream plumbing only: every byte is moved
        by cudaMemcpyAsync or by the library's conversion kernels).  For s = 0, 1, ...: upload host_ins[s], advance it one
        step (order orders[s]), download the result into host_outs[s].  All host tensors are pinned [15, nz, ny, nx]
        float32.  The grids are independent of one another, so the upload of grid s+1 (copy stream `up`, z-slabs through
        two device staging slabs, ppm_set_state from device memory) runs while grid s is downloaded (ppm_get_state into
        two more staging slabs, copy stream `down`): PCIe carries both directions at once.  Returns after the last
        download has finished (wait=False: returns once everything is enqueued; finish_host_pipelined() waits)."""
        nx, ny, nz = self.n
        step = step or self.step
        dev, main = self.device, self.stream
        if getattr(self, "_pipe", None) is None or self._pipe[0] != slab:
            mk = lambda: torch.empty((NF, slab, ny, nx), dtype=torch.float32, device=dev)
            with torch.cuda.device(dev):
                self._pipe = (slab, [mk(), mk()], [mk(), mk()], torch.cuda.Stream(dev), torch.cuda.Stream(dev))
        _, stg_in, stg_out, up, down = self._pipe
        slabs = [(z0, min(slab, nz - z0)) for z0 in range(0, nz, slab)]
        K = len(host_ins)
        in_ready, in_free, out_free = [None, None], [None, None], [None, None]
        nxt = [0, 0]                                   # (grid, slab index) of the next upload to enqueue

        def enqueue_upload():
            s, k = nxt
            if s >= K:
                return
            b = (s * len(slabs) + k) % 2
            z0, nzs = slabs[k]
            with torch.cuda.stream(up):
                if in_free[b] is not None:
                    up.wait_event(in_free[b])          # the conversion that read this staging slab is done
                for f in range(NF):
                    stg_in[b][f, :nzs].copy_(host_ins[s][f, z0:z0 + nzs], non_blocking=True)
                in_ready[b] = up.record_event()
            nxt[0], nxt[1] = (s, k + 1) if k + 1 < len(slabs) else (s + 1, 0)

        def convert_upload(s, k):
            b = (s * len(slabs) + k) % 2
            z0, nzs = slabs[k]
            main.wait_event(in_ready[b])
            self._check(lib().ppm_set_state(self._h, self._ptrs(stg_in[b][:, :nzs]), int(z0), int(nzs), 1))
            in_free[b] = main.record_event()

        with torch.cuda.device(dev):
            enqueue_upload(); enqueue_upload()
            for k in range(len(slabs)):                # grid 0 goes up alone
                convert_upload(0, k)
                enqueue_upload()
            for s in range(K):
                step(dt, orders[s])
                for k, (z0, nzs) in enumerate(slabs):
                    b = k % 2
                    if out_free[b] is not None:
                        main.wait_event(out_free[b])   # the download that read this staging slab is done
                    view = stg_out[b][:, :nzs]
                    self._check(lib().ppm_get_state(self._h, self._ptrs(view), int(z0), int(nzs), 1))
                    ev = main.record_event()
                    with torch.cuda.stream(down):
                        down.wait_event(ev)
                        for f in range(NF):
                            host_outs[s][f, z0:z0 + nzs].copy_(view[f], non_blocking=True)
                        out_free[b] = down.record_event()
                    if s + 1 < K:                      # slab k of the state is free again: the next grid's slab k moves in
                        convert_upload(s + 1, k)
                        enqueue_upload()
            if wait:
                down.synchronize()
                main.synchronize()
        if wait:
            self.sync()

    def finish_host_pipelined(self):
        """waits for a step_host_pipelined(..., wait=False) of this context (two contexts on two streams, each fed with every
        other grid, keep both directions of the link busy while either one computes) and reports the state flag"""
        if getattr(self, "_pipe", None) is not None:
            self._pipe[4].synchronize()
        self.stream.synchronize()
        self.sync()

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

    def reduce_conserved_static(self, out, nblocks=0):
        """ppm_reduce_conserved_static: the six sums into `out` (a float64 CUDA tensor of 6 elements the caller owns); the
        partial sums live in the library's static device array — no allocation, no synchronisation (enqueue only)"""
        if not (out.is_cuda and out.dtype == torch.float64 and out.numel() == 6 and out.is_contiguous()):
            raise ValueError("out: a contiguous float64 CUDA tensor of 6 elements")
        self._check(lib().ppm_reduce_conserved_static(self._h, int(nblocks), C.c_void_p(out.data_ptr())))
        return out

    def sync(self):
        self._check(lib().ppm_sync(self._h))

    def set_chunk(self, chunk):
        self._check(lib().ppm_set_chunk(self._h, int(chunk)))

    def set_option(self, option, value):
        self._check(lib().ppm_set_option(self._h, int(option), int(value)))

    def axis_path(self, axis):
        return int(lib().ppm_axis_path(self._h, int(axis)))

    def set_sphere(self, radius, center=(0.5, 0.5, 0.5)):
        """NEXT-3: confining sphere; radius <= 0 switches it off"""
        cen = (C.c_double * 3)(*[float(v) for v in center])
        self._check(lib().ppm_set_sphere(self._h, float(radius), cen))

    # ---- NEXT-4: brick decomposition (the exchange itself lives in paper_1810_13416_b200/decomposition.py) ----
    def halo_floats(self, axis):
        return int(lib().ppm_halo_floats(self.n[0], self.n[1], self.n[2], int(axis)))

    def pack_halo(self, axis, side, dst):
        """the first (side 0) / last (side 1) brick layer along `axis` -> dst (device float32 tensor of halo_floats(axis))"""
        assert dst.is_cuda and dst.dtype == torch.float32 and dst.is_contiguous() and dst.numel() >= self.halo_floats(axis)
        self._check(lib().ppm_pack_halo(self._h, int(axis), int(side), C.c_void_p(dst.data_ptr())))

    def set_halo(self, axis, side, layer):
        """registers the neighbour's brick layer (device tensor, kept alive by this object) as the ghost brick beyond that face"""
        assert layer.is_cuda and layer.dtype == torch.float32 and layer.is_contiguous() and layer.numel() >= self.halo_floats(axis)
        self._halos = getattr(self, "_halos", {})
        self._halos[(axis, side)] = layer
        self._check(lib().ppm_set_halo(self._h, int(axis), int(side), C.c_void_p(layer.data_ptr())))

    def set_origin(self, org):
        self._check(lib().ppm_set_origin(self._h, (C.c_int * 3)(*[int(v) for v in org])))

    def sweep_cfl(self, dt, axis):
        self._check(lib().ppm_sweep_cfl(self._h, float(dt), int(axis)))

    def set_two_fluid(self, gamma_tracked, gamma_rest=0.0):
        """NEXT-4: two-fluid equation of state (reading R25); gamma_tracked <= 0 switches it off"""
        self._check(lib().ppm_set_two_fluid(self._h, float(gamma_tracked), float(gamma_rest)))

    def spin_up(self, domega):
        """NEXT-3: one increment of the solid-body rotation ramp about z"""
        self._check(lib().ppm_spin_up(self._h, float(domega)))

    def measure_fp32_peak(self):
        """achieved Tflop/s of a register-only FFMA kernel on this device (bench.py's roofline.alu denominator)"""
        v = C.c_double()
        self._check(lib().ppm_measure_fp32_peak(self._h, C.byref(v)))
        return v.value

    def launch_count(self):
        return int(lib().ppm_launch_count(self._h))
