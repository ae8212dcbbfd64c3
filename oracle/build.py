"""Compile oracle/*.cpp into oracle/liboracle.so (TEST INFRASTRUCTURE ONLY).

Flags follow DESIGN.md: -O2, no FMA contraction, no fast-math, so every fp32 step of the MAC and
the key quantisation is rounded exactly as written.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "bonsai_oracle.cpp"), os.path.join(HERE, "integrator_oracle.cpp"),
        os.path.join(HERE, "refresh_oracle.cpp"), os.path.join(HERE, "mac_oracle.cpp")]
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(p) for p in SRCS)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
           "-shared", "-fPIC", *SRCS, "-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
