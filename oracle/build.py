"""Build oracle/libmo.so from oracle/mo.c (gcc, OpenMP, libquadmath).

TEST INFRASTRUCTURE: the oracle is only built/loaded by tests/, __graft_entry__ and
bench.py's cpu_baseline / --impl reference legs.  `python -m oracle.build` rebuilds it.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mo.c")
LIB = os.path.join(HERE, "libmo.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", LIB, SRC,
           "-lquadmath", "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
