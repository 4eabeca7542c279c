"""Compile the oracle (plain C) into oracle/liboracle.so.  Building the checker is not
using it: __graft_entry__.build() calls this; only tests/, smoke() and bench.py's
cpu_baseline / --impl reference legs ever load the result."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "hcc_oracle.c")
LIB = os.path.join(_HERE, "liboracle.so")

# no -march: the .so travels to another machine; no contraction, no fast-math: every
# operation is the IEEE operation the source states
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
          "-Wall", "-Wextra"]


def build(force=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    subprocess.run(["gcc", *CFLAGS, "-o", LIB + ".tmp", SRC, "-lm"], check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
