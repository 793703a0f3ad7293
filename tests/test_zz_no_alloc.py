"""GPU test of sim_qdot_pdf_noalloc, the one entry point of libnmsdt.so that never allocates device memory.

Why it exists: sim_qdot_pdf (Eq. 14-16) keeps its reduction scratch in a buffer that the handle grows
with cudaMalloc.  Two kinds of user cannot live with that: a host code that has given the whole GPU to its own memory arena
and lends the library its workspace (sim_create's device_buf) -- the driver's heap has nothing left, the call fails; and a
monitor that samples the histogram every few steps while other handles have steps queued -- cudaMalloc / cudaFree
synchronise the device and stall them.  For these the library carries a fixed ~2.3 MiB __device__ array (512 bins at most)
that every handle on a GPU shares and that keeps the previous call's contents.

What is checked: the no-alloc call returns exactly what sim_qdot_pdf returns (same kernels, same launch shape, fixed
summation order: the suite's tolerance for a repeated histogram is bit equality, tests/test_gpu_post.py), on two calls in a
row and across a change of window and of handle in between (stale contents of the shared array must not leak into a later
result); the size limit is an error with a message that names it; a warmed-up call leaves the device's free memory where it
was.  The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It builds its own states with the library alone (no oracle), so it passes alone in a fresh process, where
its first call is the one that looks up the array's address, as well as after the rest of the suite."""
import numpy as np
import pytest

from paper_1905_05727_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1905_05727_b200 import binding, build
    build.build()
    binding.load_library()
    return binding


def _reacting(B, name, steps, **kw):
    cfg = inputs.config(name, reactive=1, **kw)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    s.init(cfg["init"])
    s.step(steps)
    return s


def test_noalloc_histogram_equals_the_allocating_path_twice_in_a_row(B):
    import torch
    s1 = _reacting(B, "C1", 500)                                # 256x128, one cavity collapsing under a 9 GPa shock
    s2 = _reacting(B, "C4", 120, nx=333, ny=77)                 # ragged box of random cavities: other bins, other counts
    try:
        wide = (-30.0, 0.12, 512)                               # the largest window the static array takes; holds every reacting cell
        paper = (2.0, 0.02, 400)                                # the paper's window
        small = (0.0, 0.5, 24)
        ref = {(id(s), w): s.qdot_pdf(*w) for s in (s1, s2) for w in (wide, paper, small)}
        assert ref[(id(s1), wide)][1].sum() > 50 and ref[(id(s2), wide)][1].sum() > 50, "the states must contain reacting material"
        assert not np.array_equal(ref[(id(s1), wide)][1], ref[(id(s2), wide)][1])

        # two calls in a row, then every change that could expose leftovers: fewer bins after more, another handle, back again
        order = [(s1, wide), (s1, wide), (s1, small), (s2, paper), (s2, paper), (s1, paper), (s2, wide), (s2, small), (s1, wide)]
        for s, w in order:
            m, c = s.qdot_pdf_noalloc(*w)
            mr, cr = ref[(id(s), w)]
            assert np.array_equal(c, cr), "counts differ from sim_qdot_pdf for window %r" % (w,)
            assert np.array_equal(m, mr), "masses differ from sim_qdot_pdf for window %r" % (w,)

        # the allocating path in between does not disturb it, nor the other way round
        m, c = s1.qdot_pdf(*paper)
        assert np.array_equal(m, ref[(id(s1), paper)][0]) and np.array_equal(c, ref[(id(s1), paper)][1])
        m, c = s1.qdot_pdf_noalloc(*paper)
        assert np.array_equal(m, ref[(id(s1), paper)][0]) and np.array_equal(c, ref[(id(s1), paper)][1])

        # no device memory changes hands once the first call on this device is behind us
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for w in (wide, small, paper):
            s2.qdot_pdf_noalloc(*w)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
    finally:
        s1.close()
        s2.close()


def test_noalloc_limits_and_inert_runs(B):
    s = _reacting(B, "C1", 20)
    try:
        with pytest.raises(Exception) as ei:
            s.qdot_pdf_noalloc(2.0, 0.02, 513)                  # one bin more than the static array holds
        assert "512" in str(ei.value)
        m, c = s.qdot_pdf(2.0, 0.02, 513)                       # the allocating path takes it
        assert m.shape == (513,)
        for bad in ((2.0, 0.02, 0), (2.0, 0.0, 400), (2.0, -1.0, 400)):
            with pytest.raises(Exception):
                s.qdot_pdf_noalloc(*bad)
        m, c = s.qdot_pdf_noalloc(2.0, 0.02, 512)               # the limit itself is fine
        mr, cr = s.qdot_pdf(2.0, 0.02, 512)
        assert np.array_equal(m, mr) and np.array_equal(c, cr)
    finally:
        s.close()
    cfg = inputs.config("C1", reactive=0)                       # inert: zeros, as sim_qdot_pdf
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    try:
        with pytest.raises(Exception):
            s.qdot_pdf_noalloc()                                # not initialised
        s.init(cfg["init"])
        m, c = s.qdot_pdf_noalloc()
        assert m.sum() == 0.0 and c.sum() == 0
    finally:
        s.close()
