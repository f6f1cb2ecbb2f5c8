"""Build libnh_b200.so (the C-ABI library of include/nh_b200.h) from csrc/ with nvcc, in-tree.

    python -m paper_1706_04551_b200.build [--force]   ->  paper_1706_04551_b200/libnh_b200.so

sm_100a only (-gencode arch=compute_100a,code=sm_100a), -lineinfo for ncu's source page,
-fmad=false: fp64 arithmetic in source order, no FMA contraction (csrc/nh_internal.cuh states
the arithmetic contract).  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libnh_b200.so")
SOURCES = ["nh_api.cu", "nh_predictor.cu", "nh_pressure.cu", "nh_solver.cu"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-shared",
              "-cudart", "shared"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    d.append(os.path.join(INC, "nh_b200.h"))
    d.append(os.path.abspath(__file__))
    return d


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB):
        m = os.path.getmtime(LIB)
        if all(m >= os.path.getmtime(p) for p in _deps()):
            return LIB
    extra = os.environ.get("NH_NVCC_EXTRA", "").split()   # developer knob: extra -D switches for experiments
    cmd = [_nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
        ["-I", INC, "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
