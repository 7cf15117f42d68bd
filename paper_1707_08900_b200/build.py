"""Build libfd6.so (the C-ABI library of include/fd6.h) for sm_100a, in-tree.

Usage: python -m paper_1707_08900_b200.build [--force] [--verbose]
Called by __graft_entry__.build().  Plain nvcc, static cudart, no libtorch: the library takes device
memory and streams through the hooks of fd6.h, so it does not depend on torch's ABI.

Translation units (compiled in parallel, objects under paper_1707_08900_b200/build/, re-made only when a
dependency or the flags changed): fd6.cu (C ABI, launch sequencing, the direct kernels) and ten units of
tiled-kernel instantiations, fd6_tiled_inst.cu for each value type (float, double, V2), with and without the
forcing term, in the wide and (double, V2) the tall tile shape.
"""
import concurrent.futures
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(HERE, "..", "include")
OBJDIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libfd6.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "--expt-relaxed-constexpr",
    "-Xptxas", "-warn-spills",
]

_COMMON = ["fd6_common.cuh", "fd6_tiled_host.cuh"]
_HEADERS = [os.path.join(INCLUDE, "fd6.h"), os.path.join(INCLUDE, "fd6_testing.h")]


def units():
    """(object name, source, extra -D flags, dependencies)"""
    out = [("fd6.o", "fd6.cu", [], ["fd6.cu", "fd6_kernels_direct.cuh"] + _COMMON)]
    for t, shapes in (("V2", (1, 0)), ("double", (1, 0)), ("float", (0,))):  # longest compilations first
        for shape in shapes:
            for force in ("false", "true"):
                out.append((f"tiled_{t}_{force}_{shape}.o", "fd6_tiled_inst.cu",
                            [f"-DFD6_INST_T={t}", f"-DFD6_INST_FORCE={force}", f"-DFD6_INST_SHAPE={shape}"],
                            ["fd6_tiled_inst.cu", "fd6_kernels_tiled.cuh"] + _COMMON))
    return out


def sources():
    return [os.path.join(CSRC, "fd6.cu"), os.path.join(CSRC, "fd6_tiled_inst.cu")]


def _stale(obj, deps, stamp):
    if not os.path.exists(obj) or not os.path.exists(obj + ".flags"):
        return True
    with open(obj + ".flags") as f:
        if f.read() != stamp:
            return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    extra = os.environ.get("FD6_EXTRA_FLAGS", "").split()  # e.g. -D switches of kernel experiments
    os.makedirs(OBJDIR, exist_ok=True)
    jobs, objs = [], []
    for name, src, defs, deps in units():
        obj = os.path.join(OBJDIR, name)
        objs.append(obj)
        cmd = [NVCC] + FLAGS + extra + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
        stamp = hashlib.sha1(" ".join(cmd).encode()).hexdigest()
        dep_paths = [os.path.join(CSRC, d) for d in deps] + _HEADERS + [os.path.abspath(__file__)]
        if force or _stale(obj, dep_paths, stamp):
            jobs.append((obj, cmd, stamp))

    def compile_one(job):
        obj, cmd, stamp = job
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode == 0:
            with open(obj + ".flags", "w") as f:
                f.write(stamp)
        return obj, res

    failed = False
    with concurrent.futures.ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as pool:
        for obj, res in pool.map(compile_one, jobs):
            if verbose or res.returncode != 0:
                sys.stderr.write(f"---- {os.path.basename(obj)}\n" + res.stdout + res.stderr)
            failed = failed or res.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libfd6.so")
    if jobs or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed linking libfd6.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
