"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/ppm.h declares, validates
arguments before touching CUDA, and fails loudly (PPM_ECUDA) when there is no GPU — there is no CPU fallback."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

from paper_1810_13416_b200 import build as libbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    libbuild.build()
    from paper_1810_13416_b200 import binding
    return binding


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "ppm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ppm_[a-z0-9_]+)\s*\(", hdr))
    assert {"ppm_create", "ppm_set_state", "ppm_step", "ppm_get_state", "ppm_reduce_conserved", "ppm_cfl_dt"} <= declared
    L = lib.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(lib.EXPORTS)


def test_binding_constants_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "ppm.h")).read()
    assert int(re.search(r"#define\s+PPM_STATIC_RED_BLOCKS\s+(\d+)", hdr).group(1)) == lib.STATIC_RED_BLOCKS
    assert int(re.search(r"#define\s+PPM_NFIELDS\s+(\d+)", hdr).group(1)) == lib.NF
    assert int(re.search(r"PPM_BC_HALO\s*=\s*(\d+)", hdr).group(1)) == lib.BC_HALO


def test_struct_layout_matches_header(lib):
    # the ctypes mirror must agree with the C struct (struct_size is checked by ppm_create)
    assert C.sizeof(lib.ppm_gravity) == 72
    assert C.sizeof(lib.ppm_params) == 8 + 16 + 32 + 72 + 24 + 8


def _create(lib, **kw):
    args = dict(nx=8, ny=8, nz=8, dx=0.125, gamma=5 / 3, bc=(0,) * 6, grav=None)
    args.update(kw)
    prm, keep = lib.make_params(args["nx"], args["ny"], args["nz"], args["dx"], args["gamma"], args["bc"], args["grav"],
                                rho_floor=args.get("rho_floor", 1e-10), p_floor=args.get("p_floor", 1e-10))
    if "struct_size" in args:
        prm.struct_size = args["struct_size"]
    h = C.c_void_p()
    a, b = args.get("a", 0x1000), args.get("b", 0x2000)
    rc = lib.lib().ppm_create(C.byref(h), C.byref(prm), C.c_void_p(a), C.c_void_p(b))
    return rc, h, lib.lib().ppm_last_error(None).decode()


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    E = lib.PPM_EINVAL
    assert _create(lib, nx=0)[0] == E
    assert _create(lib, dx=0.0)[0] == E
    assert _create(lib, gamma=1.0)[0] == E
    assert _create(lib, rho_floor=0.0)[0] == E
    assert _create(lib, bc=(0, 1, 0, 0, 0, 0))[0] == E            # periodic must pair up
    assert _create(lib, bc=(0, 0, 0, 0, 7, 7))[0] == E
    assert _create(lib, nz=3, bc=(0, 0, 0, 0, 1, 1))[0] == E       # reflecting axis needs >= 4 cells
    assert _create(lib, struct_size=8)[0] == E
    assert _create(lib, a=0)[0] == E and _create(lib, a=0x1040)[0] == E and _create(lib, a=0x2000)[0] == E   # NULL, not 128-byte aligned, aliased
    tab = np.ones(5, dtype=np.float32)
    bad = dict(kind=1, s0=0.0, ds=0.1, g=tab, rho0=tab, p0=tab)    # CONST_Z table must sit on centres and faces
    rc, _, msg = _create(lib, grav=bad)
    assert rc == E and "CONST_Z" in msg
    assert _create(lib, grav=dict(kind=9, s0=0.0, ds=0.1, g=tab, rho0=tab, p0=tab))[0] == E


def test_state_floats_is_whole_brick_records(lib):
    L = lib.lib()
    assert L.ppm_state_floats(8, 8, 8) == 15 * 512
    assert L.ppm_state_floats(512, 512, 512) == 15 * 512 ** 3
    assert L.ppm_state_floats(37, 29, 23) == 15 * 64 * 10 * 8 * 6      # extents rounded up to 4-cell bricks
    assert L.ppm_state_floats(1, 1, 1) == 15 * 64
    assert L.ppm_state_floats(0, 8, 8) == 0 and L.ppm_state_floats(8, -1, 8) == 0


def test_tail_segment_plan(lib):
    """host logic of the sweep scheduling: the pencils of the ragged last wave are cut so that the wave fills the
    resident CTA slots; a cut costs 8 warm-up cells"""
    L = lib.lib()
    slots = 148 * 3
    assert L.ppm_plan_tail_chunk(2048 - 4 * slots, slots, 512) == 172        # 512^3: 272 tail tiles cut in three
    assert L.ppm_plan_tail_chunk(0, slots, 512) == 0 and L.ppm_plan_tail_chunk(5, 0, 512) == 0
    for tail in (1, 7, 100, 200, 272, 300, 443):
        for n in (32, 100, 512, 1024):
            ch = L.ppm_plan_tail_chunk(tail, slots, n)
            nch = -(-n // ch)
            assert (ch % 4 == 0 or ch == n) and 0 < ch <= max(n, 4) and (ch >= 32 or nch == 1)
            cost = -(-tail * nch // slots) * (ch + (8 if nch > 1 else 0))   # waves of segments x segment length
            assert cost <= n                                                 # never worse than marching whole pencils
    # a tail that already fills the slots is not cut
    assert L.ppm_plan_tail_chunk(slots - 1, slots, 512) == 512


def test_null_context_calls_return_einval(lib):
    L = lib.lib()
    v = C.c_double()
    assert L.ppm_step(None, 0.1, 0) == lib.PPM_EINVAL
    assert L.ppm_sweep(None, 0.1, 0) == lib.PPM_EINVAL
    assert L.ppm_cfl_dt(None, 0.8, C.byref(v)) == lib.PPM_EINVAL
    assert L.ppm_reduce_conserved(None, None) == lib.PPM_EINVAL
    assert L.ppm_sync(None) == lib.PPM_EINVAL
    assert L.ppm_reduce_conserved_static(None, 0, None) == lib.PPM_EINVAL
    assert L.ppm_set_chunk(None, 4) == lib.PPM_EINVAL
    assert L.ppm_launch_count(None) == 0
    L.ppm_destroy(None)
    assert isinstance(L.ppm_last_error(None), bytes)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_gpu_fails_loudly_no_cpu_fallback(lib):
    rc, h, msg = _create(lib)
    assert rc == lib.PPM_ECUDA and "no CPU fallback" in msg and not h.value
    with pytest.raises(RuntimeError):
        lib.PPM(8, 8, 8, 0.125, 5 / 3, (0,) * 6)


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1810_13416_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle", "").replace("oracle/", "").replace("and the oracle", "") or \
                    not re.search(r"^\s*(from|import)\s+oracle|#include\s+\".*oracle", src, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1810_13416_b200|#include\s+\"ppm", src, flags=re.M), f
