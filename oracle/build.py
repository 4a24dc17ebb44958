"""Build the oracle shared library (test infrastructure).  python -m oracle.build

Flags are part of the parity contract: -O2 -ffp-contract=off, no fast-math, so
the only fused multiply-adds are the explicit std::fma / std::fmaf calls in soax_oracle.cpp.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "soax_oracle.cpp")
LIB = os.path.join(HERE, "libsoax_oracle.so")
FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["g++", *FLAGS, SRC, "-o", tmp], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
