"""Out-of-bounds writes, found without compute-sanitizer (closed on this GPU pool: profiles/r02_sanitizers.md).

The library works inside one workspace the caller may lend it (`sim_create(device_buf, bytes)`).  Here the workspace sits
between two guard bands filled with a pattern, on ragged grids (odd nx, sizes that are multiples of no tile, rows that end
in a pair whose second cell is padding), and every call of the hot path and of the post-processing runs on it.  Afterwards
  * both guard bands still hold the pattern (nothing wrote outside the workspace);
  * inside both plane sets the padding -- columns left of the two ghost columns and right of them, which no kernel may touch --
    is still the zero `sim_create` wrote (a stray store of a row piece or of a pair would land there first);
  * the state is finite and equals the oracle's (a stray READ of padding or of another row shows up as a parity failure).
"""
import ctypes as C

import numpy as np
import pytest

from paper_1905_05727_b200 import inputs
from parity_util import TOL_ONE_STEP, rel_diff

pytestmark = pytest.mark.gpu
GUARD = 1 << 20
PATTERN = 0xA5


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1905_05727_b200 import binding, build
    build.build()
    binding.load_library()
    return binding


def _guarded(B, cfg, variant):
    import torch
    nbytes = B.workspace_bytes(cfg["grid"])
    buf = torch.full((nbytes + 2 * GUARD,), PATTERN, dtype=torch.uint8, device="cuda")
    assert buf.data_ptr() % 256 == 0
    ws = buf[GUARD:GUARD + nbytes]
    return buf, ws, B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant, workspace=ws), nbytes


def _check(B, buf, ws, sim, nbytes, what):
    import torch
    torch.cuda.synchronize()
    assert bool((buf[:GUARD] == PATTERN).all()) and bool((buf[GUARD + nbytes:] == PATTERN).all()), "%s: a write outside the workspace" % what
    info = sim.slab_info()                       # device pointers of the two plane sets, plane stride, pitch
    nx, ny, pitch, fs = sim.nx, sim.ny, info.pitch, info.plane_stride
    rows = ny + 4
    for k in range(2):
        off = int(info.plane0[k]) - ws.data_ptr()
        assert 0 <= off and off + 7 * fs * 8 <= nbytes
        planes = ws[off:off + 7 * fs * 8].view(torch.float64).view(7, fs)[:, :rows * pitch].view(7, rows, pitch)
        left, right = planes[:, :, :14], planes[:, :, 16 + nx + 2:]
        assert bool((left == 0).all()), "%s: plane set %d, a write left of the ghost columns" % (what, k)
        assert bool((right == 0).all()), "%s: plane set %d, a write right of the ghost columns (pitch %d, nx %d)" % (what, k, pitch, nx)


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("nx,ny,bcy", [(83, 37, 1), (255, 64, 0), (257, 31, 1), (2051, 5, 1), (129, 130, 2), (64, 3, 1)])
def test_nothing_is_written_outside_the_state(O, B, nx, ny, bcy, variant):
    cfg = inputs.config("C4", nx=nx, ny=ny, p_shock=9e9)
    cfg["grid"].update(bc_ylo=bcy, bc_yhi=bcy)
    cfg["init"].update(shock_cells=min(cfg["init"]["shock_cells"], nx // 3), x_lo=nx // 3, phi=0.0, ncav=0,
                       cavities=[(nx // 2, ny / 2.0, min(nx, ny) / 5.0), (nx - 3.0, 1.0, 4.0)])
    buf, ws, s, nbytes = _guarded(B, cfg, variant)
    s.init(cfg["init"])
    _check(B, buf, ws, s, nbytes, "sim_init")
    o = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=4)
    o.init(cfg["init"])
    o.step(30)
    s.init_fields(o.state())
    _check(B, buf, ws, s, nbytes, "sim_init_fields")
    for it in range(5):
        o.step(1), s.step(1)
    r = rel_diff(s.state(), o.state(), o.read_field("c"))
    assert max(r) <= 5 * TOL_ONE_STEP, r
    _check(B, buf, ws, s, nbytes, "sim_step")
    s.step(20)                                    # graph replay
    for d in (0, 1):
        s.sweep(d, 0.5 * s.cfl_dt())
    s.source(1e-10)
    s.halo(0), s.halo(1)
    s.diagnostics(), s.profiles(1.01e5), s.qdot_pdf(), s.read_field("q3"), s.cavities()
    _check(B, buf, ws, s, nbytes, "piecewise calls and post-processing")
    assert all(np.isfinite(a).all() for a in s.state())
    # derived fields are gathered densely into the idle plane set B (its padding included: documented scratch use), so
    # only the guard bands are checked after them -- and the next steps must not care what the padding of B holds
    T2 = s.read_field("T2")
    assert np.isfinite(T2).all()
    o2 = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=4)
    q = s.state()
    o2.init_fields(q)
    s.init_fields(q)
    s.read_field("p")
    for it in range(2):
        o2.step(1), s.step(1)
    r = rel_diff(s.state(), o2.state(), o2.read_field("c"))
    assert max(r) <= 5 * TOL_ONE_STEP, r           # (a sanity bound here: the parity tests proper are tests/test_gpu_parity.py)
    import torch
    torch.cuda.synchronize()
    assert bool((buf[:GUARD] == PATTERN).all()) and bool((buf[GUARD + nbytes:] == PATTERN).all())
    s.close()


def test_generator_and_painter_stay_inside(O, B):
    """seeded generator + painter on a periodic strip whose cavities straddle the top/bottom boundary and the right edge"""
    cfg = inputs.config("C5", nx=1021, ny=253)
    buf, ws, s, nbytes = _guarded(B, cfg, 1)
    s.init(cfg["init"])
    assert len(s.cavities()) > 10
    _check(B, buf, ws, s, nbytes, "sim_init (generator)")
    s.step(6)
    _check(B, buf, ws, s, nbytes, "sim_step after the generator")
    assert s.diagnostics()["bad_state"] == 0
    s.close()
