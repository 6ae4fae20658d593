"""Build oracle/liboracle.so (g++ -O2 -std=c++17 -ffp-contract=off).  TEST INFRASTRUCTURE ONLY.

The oracle is the independent CPU restatement of the paper's method (see oracle/oracle.h); it
links against nothing but libstdc++/libm and shares no source with the CUDA tree.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SOURCES = ["sampler.cpp"]
HEADERS = ["oracle.h", "models.hpp", "rng.hpp"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               "-Wall", "-Wextra", "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
        subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
