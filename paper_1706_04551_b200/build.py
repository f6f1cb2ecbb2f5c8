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
KERNEL_SOURCES = ["nh_core.cu", "nh_predictor.cu", "nh_pressure.cu", "nh_solver.cu"]  # once per precision
ABI_SOURCES = ["nh_abi.cu", "nh_peak.cu", "nh_static.cu"]   # once
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-cudart", "shared"]
OBJ = os.path.join(HERE, "build")


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
    """Every kernel file and nh_core.cu are compiled twice (-DNH_PREC=64: namespace nh64, the fp64
    contract; -DNH_PREC=32: namespace nh32, the fp32 variant), nh_abi.cu once; the objects are
    compiled in parallel and linked into one shared library."""
    if not force and os.path.exists(LIB):
        m = os.path.getmtime(LIB)
        if all(m >= os.path.getmtime(p) for p in _deps()):
            return LIB
    os.makedirs(OBJ, exist_ok=True)
    common = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-I", INC, "-c"]
    jobs = []
    for prec in (64, 32):
        for src in KERNEL_SOURCES:
            obj = os.path.join(OBJ, f"{os.path.splitext(src)[0]}_{prec}.o")
            jobs.append((obj, common + [f"-DNH_PREC={prec}", "-o", obj, os.path.join(CSRC, src)]))
    for src in ABI_SOURCES:
        obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
        jobs.append((obj, common + ["-o", obj, os.path.join(CSRC, src)]))
    procs = [(o, subprocess.Popen(cmd, cwd=HERE, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
             for o, cmd in jobs]
    failed = []
    for o, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(f"--- {os.path.basename(o)}\n{out}")
        if pr.returncode != 0:
            failed.append(o)
    if failed:
        raise subprocess.CalledProcessError(1, "nvcc -c", output=", ".join(failed))
    subprocess.run([_nvcc(), "-shared", "-cudart", "shared", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-o", LIB] + [o for o, _ in jobs], check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
