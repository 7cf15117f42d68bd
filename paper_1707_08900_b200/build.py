"""Build libfd6.so (the C-ABI library of include/fd6.h) for sm_100a, in-tree.

Usage: python -m paper_1707_08900_b200.build [--force] [--verbose]
Called by __graft_entry__.build().  Plain nvcc, static cudart, no libtorch: the library takes device
memory and streams through the hooks of fd6.h, so it does not depend on torch's ABI.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfd6.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "--expt-relaxed-constexpr",
    "-Xptxas", "-warn-spills",
]


def sources():
    return [os.path.join(CSRC, "fd6.cu")]


def _deps():
    return glob.glob(os.path.join(CSRC, "*")) + [os.path.join(HERE, "..", "include", "fd6.h"), os.path.abspath(__file__)]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    extra = os.environ.get("FD6_EXTRA_FLAGS", "").split()  # e.g. -D switches of kernel experiments
    cmd = [NVCC] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + sources()
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libfd6.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
