"""Device check of the fused kernels' own fp64 elementary functions through the C ABI (sim_probe_math)."""
import pytest

from math_cases import check

pytestmark = pytest.mark.gpu


def test_elementary_functions_device():
    from paper_1905_05727_b200 import binding, build, inputs
    build.build()
    cfg = inputs.config("C1")
    s = binding.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    try:
        out = check(lambda fn, x, a, b: s.probe_math(fn, x, a, b))
        print(out)
    finally:
        s.close()
