"""Compile the oracle's C core (TEST INFRASTRUCTURE ONLY; see oracle/__init__.py).

gcc -O2 -ffp-contract=off (no FMA contraction) -fopenmp -shared.
Building the checker is not using it: __graft_entry__.build() may call this.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "forcefield.c")
LIB = os.path.join(HERE, "liboracle_forcefield.so")


def build(force=False):
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
