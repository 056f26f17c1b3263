"""Build step for the CPU oracle (test infrastructure): gcc -O2 -fopenmp -ffp-contract=off -> oracle/liboracle.so.
Building the checker is not using it: __graft_entry__.build() calls this; only tests/, smoke() and bench.py's
cpu_baseline / --impl reference legs ever load the result."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.c")
LIB = os.path.join(HERE, "liboracle.so")


def build(force=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall",
           "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
