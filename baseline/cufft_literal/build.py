"""Build the cuFFT-backed reference point (baseline/cufft_literal/cufft_literal.cu -> libcufft_literal.so, in-tree)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cufft_literal.cu")
LIB = os.path.join(HERE, "libcufft_literal.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    subprocess.check_call([nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                           "-Xcompiler", "-fPIC", "-shared", "-o", LIB, SRC, "-lcufft"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
