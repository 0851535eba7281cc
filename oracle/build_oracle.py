"""Build oracle/liboracle.so (TEST INFRASTRUCTURE).  Usage: python oracle/build_oracle.py [--force]

Plain g++ -O2 -fopenmp; deliberately NOT tuned (no -march=native, no -ffast-math): the oracle is the
reference for correctness and the reported CPU baseline "as it stands".
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "oracle_capi.cpp")]
DEPS = SRC + [os.path.join(HERE, f) for f in ("mhd_oracle.hpp", "tracers_oracle.hpp", "oracle.h")]
OUT = os.path.join(HERE, "liboracle.so")


def needs_build() -> bool:
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    return any(os.path.getmtime(p) > t for p in DEPS)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", OUT + ".tmp"] + SRC
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(OUT + ".tmp", OUT)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
