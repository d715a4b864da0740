"""Builds oracle/liboracle.so (host only, g++ -O2 -fopenmp; no -march=native: the built library travels to
another host). TEST INFRASTRUCTURE."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qss_oracle.cpp")
SRC_NEWTON = os.path.join(HERE, "qss_newton_oracle.cpp")
HDR = os.path.join(HERE, "qss_oracle.h")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(SRC_NEWTON), os.path.getmtime(HDR)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    # -ffp-contract=off: the oracle is the plain definition, operation by operation (no fused multiply-add)
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-fPIC", "-shared",
           "-o", tmp, SRC, SRC_NEWTON, "-lquadmath"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
