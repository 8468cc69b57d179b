"""Compile the fp64 CPU oracle (oracle/rte_oracle.cpp) into oracle/librte_oracle.so.

The oracle is TEST INFRASTRUCTURE: building it here is not using it.  Run as a script or call build().
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "rte_oracle.cpp")
LIB = os.path.join(HERE, "librte_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
