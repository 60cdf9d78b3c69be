"""TEST INFRASTRUCTURE — builds the CPU oracle (oracle/liboracle.so) with g++.

Plain IEEE arithmetic: no -ffast-math, no FMA contraction, so that what the oracle
computes is the formula as written.  `python oracle/build.py` or `oracle.build.build()`.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SOURCES = ["capi.cpp"]
HEADERS = ["philox.hpp", "dual.hpp", "scene.hpp", "path.hpp", "analytic2d.hpp", "samplers.hpp", "bias.hpp"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False) -> str:
    if force or stale():
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               "-Wall", "-Wextra", "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
        subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
