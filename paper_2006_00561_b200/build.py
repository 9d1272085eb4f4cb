"""Build libpa_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2006_00561_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpa_b200.so")
SOURCES = [os.path.join(CSRC, "pa_b200.cu"), os.path.join(CSRC, "pa_static.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("pa_common.cuh", "pa_sweep.cuh", "pa_resample.cuh", "pa_observe.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "pa_b200.h")]

NVCC_FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "-shared",
              "-Xcompiler", "-fPIC,-O2,-Wall", "--expt-relaxed-constexpr"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
