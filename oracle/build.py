"""Build liboracle.so (TEST INFRASTRUCTURE -- see nmsdt_oracle.h).

g++ -O2 -ffp-contract=off: no FMA contraction, so every decision in the oracle is taken on
exactly rounded operations.  -fopenmp only parallelises the row loops (results bit-identical
for any thread count); the default is one thread.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SRC = [os.path.join(HERE, "nmsdt_oracle.cpp")]
HDR = [os.path.join(HERE, "nmsdt_oracle.h")]


def build(force: bool = False) -> str:
    deps = SRC + HDR
    if (not force) and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", LIB] + SRC
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
