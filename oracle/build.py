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
    """ORACLE_SANITIZE=1 in the environment: build with -fsanitize=address,undefined instead (same file name, so force a
    rebuild before and after), for one run of the oracle tests under the sanitizers:
        ORACLE_SANITIZE=1 python -m oracle.build
        LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 python -m pytest tests/test_oracle_*.py -q
        python -m oracle.build
    (the runtime must be preloaded because the interpreter itself is not instrumented; leak detection is off because
    CPython does not free everything at exit).  DESIGN.md section 4 records the outcome."""
    sanitize = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
    if (not force) and (not sanitize) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] if sanitize else ["-O2"]
    cmd = ["gcc"] + opt + ["-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
                           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
