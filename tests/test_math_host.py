"""Host-side check of nmsdt_math.cuh (the fused kernels' fp64 rcp / sqrt / log / pow / exp): the header compiles for
the host with emulated 20-bit seeds, so the table and polynomial logic is checked against long-double library
routines without a GPU.  The device run of the same cases is tests/test_gpu_math.py."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from math_cases import check

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def lib(tmp_path_factory):
    cuda_inc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "include")
    if not os.path.exists(os.path.join(cuda_inc, "cuda_runtime.h")):
        pytest.skip("CUDA headers not found")
    so = str(tmp_path_factory.mktemp("mathhost") / "libmathhost.so")
    subprocess.run(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-shared", "-fPIC", "-I", cuda_inc, "-o", so,
                    os.path.join(HERE, "math_host_harness.cpp")], check=True)
    L = C.CDLL(so)
    dp = C.POINTER(C.c_double)
    L.math_probe.restype = C.c_int
    L.math_probe.argtypes = [C.c_int, dp, C.c_int, C.c_double, C.c_double, dp, dp]
    return L


def test_elementary_functions_host(lib):
    dp = C.POINTER(C.c_double)

    def probe(fn, x, a, b):
        x = np.ascontiguousarray(x, dtype=np.float64)
        y0, y1 = np.empty_like(x), np.empty_like(x)
        assert lib.math_probe(fn, x.ctypes.data_as(dp), x.size, a, b, y0.ctypes.data_as(dp), y1.ctypes.data_as(dp)) == 0
        return y0, y1

    out = check(probe)
    print(out)
