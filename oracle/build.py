"""ORACLE — TEST INFRASTRUCTURE ONLY.

Builds oracle/liboracle_ref.so from the C++ sources in this directory with the host compiler
(no CUDA).  `-ffp-contract=off` gives defined fp64 arithmetic.
Building the checker is not using it: __graft_entry__.build() calls this; only tests/,
smoke() and bench.py's cpu_baseline / --impl reference legs load the result.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["oracle_api.cpp", "me_tier0.cpp", "me_tier1.cpp", "me_tier1g.cpp", "me_qed.cpp", "phase_space_ref.cpp", "vegas_ref.cpp"]
HEADERS = ["algebra.hpp", "wavefunctions.hpp", "process.hpp", "me_ref.hpp", "oracle_ref.h"]
LIB = os.path.join(HERE, "liboracle_ref.so")


def build(force: bool = False) -> str:
    deps = [os.path.join(HERE, f) for f in SOURCES + HEADERS]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
           "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
