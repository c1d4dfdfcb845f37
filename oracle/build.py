"""Build the CPU oracle (TEST INFRASTRUCTURE, not the product) with gcc.

Two shared libraries from the one source oracle/qcd_oracle.c:
  liborc.so      serial   - the definition
  liborc_omp.so  -fopenmp - site loops in parallel, reductions still serial and ordered
Run:  python oracle/build.py
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qcd_oracle.c")
LIB_SERIAL = os.path.join(HERE, "liborc.so")
LIB_OMP = os.path.join(HERE, "liborc_omp.so")


def _stale(lib):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in ("qcd_oracle.c", "qcd_oracle.h"))


def build(force=False, verbose=False):
    base = ["gcc", "-std=gnu11", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-Wno-unknown-pragmas", "-fno-fast-math",
            "-ffp-contract=off", SRC, "-lm"]
    for lib, extra in ((LIB_SERIAL, []), (LIB_OMP, ["-fopenmp"])):
        if force or _stale(lib):
            cmd = base + extra + ["-o", lib]
            if verbose:
                print(" ".join(cmd))
            subprocess.check_call(cmd)
    return LIB_SERIAL, LIB_OMP


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
