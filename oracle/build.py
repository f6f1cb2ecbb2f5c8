"""Build the CPU oracle shared library (test infrastructure, not the product).

    python -m oracle.build        ->  oracle/libnh_oracle.so

gcc -O2 -ffp-contract=off (no FMA contraction: plain IEEE fp64 arithmetic in source order),
OpenMP over rows only.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nh_oracle.c")
HDR = os.path.join(HERE, "nh_oracle.h")
LIB = os.path.join(HERE, "libnh_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        m = os.path.getmtime(LIB)
        if m >= os.path.getmtime(SRC) and m >= os.path.getmtime(HDR):
            return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
