"""Build the CPU oracle (test infrastructure) into oracle/librtvd_oracle.so with g++.

`-O2 -ffp-contract=off`: no FMA contraction, so the rounding is the one the source states.
Run as `python -m oracle.build` or through `__graft_entry__.build()`.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "rtvd_oracle.cpp")
LIB = os.path.join(HERE, "librtvd_oracle.so")


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB + ".tmp%d" % os.getpid(), SRC]      # per process: concurrent builders do not collide
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp%d" % os.getpid(), LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
