"""Build the CPU oracle (oracle/liblbm_oracle.so).  TEST INFRASTRUCTURE, NOT PRODUCT.

Flags matter for parity: `-ffp-contract=off` so the compiler never fuses a*b+c on its own (the only
fused operations are the explicit std::fma calls, which `-mfma` turns into hardware FMAs -- correctly
rounded either way), no fast-math, IEEE division.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["codecs.cpp", "lbm.cpp"]
LIB = os.path.join(HERE, "liblbm_oracle.so")
FLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
         "-mfma", "-Wall", "-Wextra"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = SOURCES + ["oracle.h", "build.py"]
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in deps)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["g++"] + FLAGS + [os.path.join(HERE, s) for s in SOURCES] + ["-o", LIB]
        subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
