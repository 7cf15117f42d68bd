"""Build the CPU oracle (test infrastructure) into oracle/libfd_oracle.so.

Usage: python oracle/build.py            (also called by __graft_entry__.build())

Flags follow DESIGN.md "Oracle": -O2, no FMA contraction, no fast-math, OpenMP for the
one `parallel for` over k-planes.  Building the checker is not using it: nothing in
the product path loads the result.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fd_oracle.cpp")
LIB = os.path.join(HERE, "libfd_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
