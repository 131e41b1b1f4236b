"""Build step for the CPU oracle (test infrastructure only; see gtbo.h).

`python -m oracle.build` compiles oracle/*.cpp into oracle/libgtbo.so with g++.
Flags: -O2 -ffp-contract=off (no FMA contraction: the neighbour test of
SURVEY.md sec. 8(c) C2 fixes the evaluation order of r^2) and OpenMP.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["gtbo_hamiltonian.cpp", "gtbo_kpm.cpp", "gtbo_vac.cpp", "gtbo_sk.cpp", "gtbo_mlp.cpp", "gtbo_spd.cpp"]
LIB = os.path.join(HERE, "libgtbo.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = SOURCES + ["gtbo.h"]
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in deps)


def build(force: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC",
           "-shared", "-Wall", "-Wextra", "-o", LIB + ".tmp"]
    cmd += [os.path.join(HERE, s) for s in SOURCES]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
