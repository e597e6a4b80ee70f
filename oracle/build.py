"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not product).

    python -m oracle.build

Compiles oracle/spin_oracle.cpp with g++ into oracle/liboracle.so.  Flags matter:
-ffp-contract=off keeps every fp32 operation separately rounded, in the order the
source states (R-14); no -ffast-math, no -march flags.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "spin_oracle.cpp")
HDR = os.path.join(HERE, "spin_oracle.h")
LIB = os.path.join(HERE, "liboracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-Wall", "-Wextra"]


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in (SRC, HDR))


def build(force: bool = False) -> str:
    if force or is_stale():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++", *FLAGS, "-o", tmp, SRC]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
