"""Build the CPU oracle (test infrastructure) into oracle/libmco.so with g++.

Building the checker is not using it: __graft_entry__.build() calls this so the
GPU box has the library; only tests/, smoke() and bench.py's cpu_baseline leg load it.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mco.cpp")
HDR = os.path.join(HERE, "mco.h")
LIB = os.path.join(HERE, "libmco.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           SRC, "-o", LIB]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
