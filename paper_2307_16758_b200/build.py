"""Builds the CUDA library in-tree:  python -m paper_2307_16758_b200.build [--force] [--verbose]

nvcc cross-compiles for sm_100a without a GPU.  The host set-up (host_mesh.cpp) is compiled with
-ffp-contract=off so the mesh geometry is the literal IEEE evaluation of its formulas; OpenMP only
spreads its independent per-cell / per-edge loops over the host cores (set-up time, not results).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libswe_b200.so")
SRCS = ["swe_api.cu", "host_mesh.cpp", "host_inspect.cpp"]
DEPS = SRCS + ["swe_kernels.cuh", "swe_zone_kernels.cuh", "host_mesh.hpp", os.path.join("..", "..", "include", "swe_b200.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
EXTRA = os.environ.get("SWE_NVCC_EXTRA", "").split()   # e.g. -DSWE_FLUX_MINB=4 for tuning sweeps


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, d) for d in DEPS]
    missing = [d for d in deps if not os.path.exists(d)]
    if missing:
        # a stale library next to an incomplete source tree must not be picked up silently
        raise FileNotFoundError("paper_2307_16758_b200: source file(s) missing, cannot tell whether %s is current: %s"
                                % (os.path.basename(LIB), ", ".join(os.path.relpath(m, HERE) for m in missing)))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    objs = [os.path.join(CSRC, "%s.%d.o" % (n, os.getpid())) for n in ("host_mesh", "host_inspect")]
    cmds = [["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-Wall", "-c",
             os.path.join(CSRC, n + ".cpp"), "-o", o]
            for n, o in zip(("host_mesh", "host_inspect"), objs)]
    cmds.append([NVCC] + ARCH + ["-lineinfo", "-O3", "-std=c++17", "-shared", "-Xcompiler", "-fPIC",
                                 "-Xptxas", "-v" if verbose else "-O3"] + EXTRA + [
                                 os.path.join(CSRC, "swe_api.cu")] + objs + ["-o", tmp, "-lcudart", "-lgomp"])
    try:
        for cmd in cmds:
            if verbose:
                print(" ".join(cmd))
            subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    finally:
        for f in objs + [tmp]:
            if os.path.exists(f):
                os.remove(f)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
