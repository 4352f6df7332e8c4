"""Build the CPU oracle (test infrastructure) into oracle/libsphref.so.

g++ -O2 -ffp-contract=off: the oracle's binary32 arithmetic is exactly what the source spells
(the only fused operations are its explicit fmaf calls).  OpenMP over the outer index only.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["ref_sim.cpp", "ref_mc.cpp"]
LIB = os.path.join(HERE, "libsphref.so")


def build(force: bool = False) -> str:
    srcs = [os.path.join(HERE, s) for s in SOURCES]
    deps = srcs + [os.path.join(HERE, "ref.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB] + srcs + ["-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
