"""Build the CPU oracle shared library (test infrastructure; see cel_oracle.cpp header).

g++ -O2 -ffp-contract=off -fopenmp: no FMA contraction, no fast-math, so the arithmetic is exactly
the sequence of IEEE operations written in the source.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cel_oracle.cpp")
LIB = os.path.join(HERE, "libcel_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", "-Wall", SRC, "-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
