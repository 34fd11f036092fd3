"""Build the fp64 CPU oracle (TEST INFRASTRUCTURE) into oracle/libppm_oracle.so with gcc.

`python -m oracle.build` or `oracle.build.build()`; __graft_entry__.build() calls it too
(building the checker is not using it).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ppm_oracle.c")
LIB = os.path.join(HERE, "libppm_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-ffp-contract=off", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
