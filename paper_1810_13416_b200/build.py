"""Build libppm_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

`python -m paper_1810_13416_b200.build [--verbose]`; __graft_entry__.build() calls build().
nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libppm_b200.so")
SOURCES = ["ppm_api.cu", "ppm_sweep.cu", "ppm_aux.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _deps():
    deps = [os.path.join(CSRC, s) for s in SOURCES]
    deps += [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    deps.append(os.path.join(ROOT, "include", "ppm.h"))
    return deps


def build(force: bool = False, verbose: bool = False, poison: bool = False) -> str:
    """poison=True: the debug variant libppm_b200_poison.so (-DPPM_DEBUG_POISON: dead ring slots of the bulk-staged sweeps
    are filled with NaN before they are refilled, so a read that races a bulk copy shows up as NaN in the parity tests);
    load it with PPM_B200_LIB=<path>."""
    LIB = globals()["LIB"] if not poison else os.path.join(HERE, "libppm_b200_poison.so")
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    cmd = [NVCC, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-ftz=true",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", LIB] + (["-DPPM_DEBUG_POISON"] if poison else []) + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="--verbose" in sys.argv, poison="--poison" in sys.argv))
