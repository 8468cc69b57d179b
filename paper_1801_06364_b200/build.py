"""Build the CUDA library (csrc/rte_lib.cu -> librte_b200.so, in-tree) for sm_100a with nvcc.

nvcc cross-compiles without a GPU.  Run `python paper_1801_06364_b200/build.py [--force] [-v]` (as a script, so the package — which refuses to import without the library — is not imported first)` or call build().
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librte_b200.so")
SOURCES = ["rte_lib.cu"]
DEPS = ["rte_lib.cu", "rte_pass.cuh", "rte_fft.cuh", "rte_tables.h", os.path.join("..", "..", "include", "rte.h")]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
