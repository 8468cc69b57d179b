"""Build the exchange micro-benchmark (tests/microbench/exchange_bench.cu -> tests/microbench/exchange_bench, in-tree)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "exchange_bench.cu")
EXE = os.path.join(HERE, "exchange_bench")


def build(force: bool = False) -> str:
    if not force and os.path.exists(EXE) and os.path.getmtime(EXE) >= os.path.getmtime(SRC):
        return EXE
    nvcc = os.environ.get("NVCC", "nvcc")
    subprocess.check_call([nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", SRC, "-o", EXE])
    return EXE


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
