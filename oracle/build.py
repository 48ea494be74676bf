"""Build the CPU oracle shared library (oracle/libraf_ref.so) with g++.

TEST INFRASTRUCTURE.  Flags are part of the oracle's definition (DESIGN.md
section 3): every fp32 coordinate operation is individually rounded, so no contraction and no
fast-math; x86-64 SSE2 arithmetic has no excess precision.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "raf_ref.cpp")
LIB = os.path.join(HERE, "libraf_ref.so")
OPS_SRC = os.path.join(HERE, "ops_ref.cpp")      # RoIPool-max, NMS, Soft-NMS
OPS_LIB = os.path.join(HERE, "libops_ref.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared"]


def _build_one(src: str, lib: str, force: bool) -> str:
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(src)
            and os.path.getmtime(lib) >= os.path.getmtime(__file__)):
        return lib
    cmd = ["g++"] + FLAGS + [src, "-o", lib + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(lib + ".tmp", lib)
    return lib


def build(force: bool = False) -> str:
    _build_one(OPS_SRC, OPS_LIB, force)
    return _build_one(SRC, LIB, force)


def build_ops(force: bool = False) -> str:
    return _build_one(OPS_SRC, OPS_LIB, force)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
