"""Builds the oracle shared library (test infrastructure; see orc_main.cpp header).

    python oracle/build.py

g++ -O2, strict IEEE (no contraction, no fast-math): the fp32 attenuation contract (DESIGN.md
R20) depends on it.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liborc.so")
SRC = [os.path.join(HERE, "orc_main.cpp")]
DEPS = SRC + [os.path.join(HERE, "orc_physics.h"), os.path.join(HERE, "orc_gs.h")]


def build(force=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in DEPS):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-shared", "-fPIC",
           "-o", LIB] + SRC
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
