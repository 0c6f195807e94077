"""Build libbirkhoff4.so (csrc/birkhoff4.cu -> paper_2606_07574_b200/libbirkhoff4.so) with nvcc for sm_100a.

In-tree and explicit: `python -m paper_2606_07574_b200.build [--force]`.  nvcc cross-compiles without a GPU.
The library has no torch dependency; cudart is linked statically.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "birkhoff4.cu"), os.path.join(CSRC, "birkhoff_ot.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("bk4_math.cuh", "bk4_solve.cuh", "bk4_lean.cuh", "bk4_guarded.cuh", "bk4_project.cuh", "bk_ot.cuh", "bk4_mix.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", f) for f in ("birkhoff4.h", "birkhoff_ot.h")]
LIB = os.path.join(HERE, "libbirkhoff4.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-ftz=true",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    extra = ["-DBK4_EXPERIMENTS"] if os.environ.get("BK4_EXPERIMENTS") else []   # measurement hooks; never in the default build
    cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB + ".tmp"] + SOURCES
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
