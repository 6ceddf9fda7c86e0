"""ORACLE — TEST INFRASTRUCTURE ONLY.  Builds oracle/liboracle.so (plain C++17, g++ -O2 -ffp-contract=off).

    python oracle/build.py            # serial + OpenMP pointwise loops (results identical for any thread count)
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["apply.cpp", "rbsor.cpp", "krylov.cpp", "vcycle.cpp", "mgv.cpp", "multipole.cpp", "capi.cpp"]
HEADERS = ["grid.hpp", "solvers.hpp"]
LIB = os.path.join(HERE, "liboracle.so")


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS + ["build.py"])


def build(force=False):
    if not force and not needs_build():
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
