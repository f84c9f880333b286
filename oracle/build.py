"""Compile the CPU oracle (oracle/phx_oracle.cpp) into oracle/liboracle.so.

TEST INFRASTRUCTURE, NOT PRODUCT.  Plain g++, -O2, no FMA contraction, no fast-math, no OpenMP.
build_omp() compiles the SAME source with -fopenmp into oracle/liboracle_omp.so: the all-host-cores leg of bench.py's
cpu_baseline; the parity oracle stays the single-threaded liboracle.so.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "phx_oracle.cpp")
HDR = os.path.join(HERE, "phx_oracle.h")
LIB = os.path.join(HERE, "liboracle.so")
LIB_OMP = os.path.join(HERE, "liboracle_omp.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-Wno-unknown-pragmas", "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


def build_omp(force: bool = False) -> str:
    """The same source with the OpenMP pragmas honoured (bench.py's all-cores cpu_baseline leg only)."""
    if not force and os.path.exists(LIB_OMP):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB_OMP) >= newest:
            return LIB_OMP
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB_OMP, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB_OMP


if __name__ == "__main__":
    print(build(force=True))
    print(build_omp(force=True))
