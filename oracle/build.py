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
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)
            and os.path.getmtime(LIB) >= os.path.getmtime(__file__)):
        return LIB
    cmd = ["g++"] + FLAGS + [SRC, "-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
