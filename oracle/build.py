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
    """ORACLE_SANITIZE=1 builds and returns liboracle_san.so instead: the same source under AddressSanitizer and
    UndefinedBehaviorSanitizer (run python with LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0;
    profiles/r02_sanitizers.md)."""
    san = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
    lib = os.path.join(HERE, "liboracle_san.so") if san else LIB
    deps = SRC + HDR + [os.path.abspath(__file__)]
    if (not force) and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps):
        return lib
    opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] if san else ["-O2"]
    cmd = ["g++", "-std=c++17"] + opt + ["-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
                                         "-Wall", "-Wextra", "-o", lib] + SRC
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force=True))
