"""Host logic of the x-slab decomposition (paper_1905_05727_b200/slab.py) on CPU: the
column partition, the neighbour / boundary-kind rules, and -- with world_size 2 and 3 under gloo -- the exchange
order, the sides, the ghost placement and the max-allreduce of DistSlab, driven through a stand-in for the sim_slab_*
calls (tests/slab_standin.py; the real calls need a GPU and are checked by tests/test_gpu_slab.py).  The decomposed run
must reproduce the undivided stand-in run bit for bit."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_1905_05727_b200 import slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_covers_domain():
    for nx, w in ((10, 3), (4096, 8), (7, 3), (32768, 5), (4, 2)):
        parts = slab.partition(nx, w)
        assert parts[0][0] == 0 and sum(n for _, n in parts) == nx
        assert all(parts[r][0] + parts[r][1] == parts[r + 1][0] for r in range(w - 1))
        assert max(n for _, n in parts) - min(n for _, n in parts) <= 1 and min(n for _, n in parts) >= 2
    with pytest.raises(ValueError):
        slab.partition(5, 3)


def test_neighbours_and_boundary_kinds():
    assert slab.neighbours(0, 1, True) == (None, None)
    assert slab.neighbours(0, 4, False) == (None, 1) and slab.neighbours(3, 4, False) == (2, None)
    assert slab.neighbours(0, 4, True) == (3, 1) and slab.neighbours(3, 4, True) == (2, 0)
    assert slab.neighbours(0, 2, True) == (1, 1)
    g = dict(nx=100, ny=8, dx=1.0, dy=1.0, bc_xlo=3, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)
    g0, x0 = slab.slab_grid(g, 0, 3)
    g1, x1 = slab.slab_grid(g, 1, 3)
    g2, x2 = slab.slab_grid(g, 2, 3)
    assert (g0["bc_xlo"], g0["bc_xhi"], x0, g0["nx"]) == (3, 4, 0, 34)         # the global x-lo kind stays on rank 0
    assert (g1["bc_xlo"], g1["bc_xhi"], x1, g1["nx"]) == (4, 4, 34, 33)
    assert (g2["bc_xlo"], g2["bc_xhi"], x2, g2["nx"]) == (4, 0, 67, 33)
    gp = dict(g, bc_xlo=1, bc_xhi=1)
    assert all(slab.slab_grid(gp, r, 2)[0]["bc_xlo"] == 4 and slab.slab_grid(gp, r, 2)[0]["bc_xhi"] == 4 for r in range(2))
    assert slab.slab_grid(gp, 0, 1)[0]["bc_xlo"] == 1                           # one slab: the ordinary periodic halo


WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r); sys.path.insert(0, os.path.join(%(root)r, "tests"))
import numpy as np
import torch.distributed as dist
from paper_1905_05727_b200 import slab
from slab_standin import StandInSim
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
out = sys.argv[1]
for case, (bcx, nx, dt_fixed) in enumerate([((0, 0), 41, 0.0), ((1, 1), 36, 0.0), ((0, 0), 40, 0.01)]):
    grid = dict(nx=nx, ny=6, dx=1.0, dy=1.0, bc_xlo=bcx[0], bc_xhi=bcx[1], bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)
    ds = slab.DistSlab(grid, StandInSim, dist, "cpu", transport="staged")
    ds.init(dict(bump=3.0))
    ds.step(5, dt_fixed=dt_fixed)
    d = ds.diagnostics()
    np.savez(os.path.join(out, "case%%d_rank%%d.npz" %% (case, rank)), u=ds.sim.state(), x0=ds.x0, t=d["t"], mass=d["mass1"],
             smax=d["smax"], step=d["step"])
    ds.close()
dist.destroy_process_group()
"""


def _reference(bcx, nx, dt_fixed):
    from slab_standin import StandInSim
    grid = dict(nx=nx, ny=6, dx=1.0, dy=1.0, bc_xlo=bcx[0], bc_xhi=bcx[1], bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)
    s = StandInSim(grid)
    s.init(dict(bump=3.0), 0)
    s.slab_begin(dt_fixed)
    s.slab_ctl(0)
    for _ in range(5):
        for p in (1, 2):
            s.slab_pass(p)
        s.slab_ctl(1)
    return s


@pytest.mark.parametrize("world,port", [(2, 29621), (3, 29622)])
def test_distslab_matches_undivided_run_gloo(tmp_path, world, port):
    w = tmp_path / "worker.py"
    w.write_text(WORKER % dict(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                        "--master-addr", "127.0.0.1", "--master-port", str(port), str(w), str(tmp_path)],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    for case, (bcx, nx, dt_fixed) in enumerate([((0, 0), 41, 0.0), ((1, 1), 36, 0.0), ((0, 0), 40, 0.01)]):
        ref = _reference(bcx, nx, dt_fixed)
        parts = [np.load(tmp_path / ("case%d_rank%d.npz" % (case, rk))) for rk in range(world)]
        assert [int(p["x0"]) for p in parts] == [x0 for x0, _ in slab.partition(nx, world)]
        u = np.concatenate([p["u"] for p in parts], axis=2)
        assert np.array_equal(u, ref.state())                          # bit for bit: same dt on every rank, right ghosts
        for p in parts:                                                # every rank reports the global diagnostics
            assert float(p["t"]) == ref.t and int(p["step"]) == 5
            assert abs(float(p["mass"]) - ref.diagnostics()["mass1"]) <= 1e-12 * abs(ref.diagnostics()["mass1"])
            assert float(p["smax"]) == ref.diagnostics()["smax"]


def test_standin_detects_a_wrong_exchange():
    """the stand-in update is sensitive to the ghost columns: leaving them stale changes the result"""
    from slab_standin import StandInSim
    ref = _reference((0, 0), 41, 0.0).state()
    grid = dict(nx=41, ny=6, dx=1.0, dy=1.0, bc_xlo=0, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)
    sims = []
    for rk in range(2):
        g, x0 = slab.slab_grid(grid, rk, 2)
        s = StandInSim(g)
        s.init(dict(bump=3.0), x0)
        sims.append(s)
    for s in sims:
        s.slab_begin(0.0)
    m = max(int(s.word[0]) for s in sims)
    for s in sims:
        s.word[0] = m
        s.slab_ctl(0)
    for _ in range(5):                          # no exchange at all
        for p in (1, 2):
            for s in sims:
                s.slab_pass(p)
        m = max(int(s.word[0]) for s in sims)
        for s in sims:
            s.word[0] = m
            s.slab_ctl(1)
    assert not np.array_equal(np.concatenate([s.state() for s in sims], axis=2), ref)
