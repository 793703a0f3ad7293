"""GPU tests of the x-slab decomposition (include/nmsdt.h sim_slab_*, paper_1905_05727_b200/slab.py; SURVEY.md 8(e),
NEXT-4).  One GPU is all there is, so the decomposed step is checked in two ways that need no second device:
  * LocalSlabs: K slabs of one domain in one process, both transports (peer stores / pack-unpack), against the
    undivided run -- bit for bit, because every slab runs the same kernels with the same dt on the same stencil inputs;
  * DistSlab under torchrun with two processes sharing the GPU (gloo carries the collectives; the peer transport maps the
    other process's workspace with CUDA IPC): the multi-process plumbing end to end.  No kernel waits for another.
and once directly against the oracle (the parity gate of the other GPU tests, here on the decomposed path)."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_1905_05727_b200 import inputs
from parity_util import TOL_ONE_STEP, l1_rel, rel_diff

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1905_05727_b200 import binding, build
    build.build()
    binding.load_library()
    return binding


def _periodic_x_case():
    cfg = inputs.config("C1", nx=192, ny=96)
    cfg["grid"].update(bc_xlo=inputs.BC_PERIODIC, bc_xhi=inputs.BC_PERIODIC, bc_ylo=inputs.BC_PERIODIC, bc_yhi=inputs.BC_PERIODIC)
    # cavities on the inner seams of 2 and 3 slabs; no shocked slab (the test adds a pressure pulse on the wrap-around seam)
    cfg["init"].update(shock_cells=0, cavities=[(97.0, 70.0, 10.0), (62.0, 30.0, 9.0), (20.0, 50.0, 8.0)])
    return cfg


CASES = {
    "C1": lambda: inputs.config("C1"),                                   # cavity (80..112) straddles the seam of 3 slabs at column 86
    "C4crop": lambda: inputs.config("C4", nx=1024, ny=256),             # seeded generator, periodic y, shock in slab 0
    "C5crop-inert-mc": lambda: _mc(inputs.config("C5", nx=768, ny=256, reactive=0)),
    "periodic-x": _periodic_x_case,
}


def _mc(cfg):
    cfg["grid"]["limiter"] = inputs.LIM_MC
    return cfg


@pytest.mark.parametrize("case,k,transport,steps", [("C1", 3, "peer", 60), ("C1", 2, "staged", 60), ("C4crop", 3, "peer", 40),
                                                    ("C4crop", 4, "staged", 25), ("C5crop-inert-mc", 3, "peer", 30),
                                                    ("periodic-x", 2, "peer", 40), ("periodic-x", 3, "staged", 40)])
def test_local_slabs_equal_the_undivided_run_bit_for_bit(B, case, k, transport, steps):
    from paper_1905_05727_b200 import slab
    cfg = CASES[case]()
    one = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    one.init(cfg["init"])
    many = slab.LocalSlabs(cfg["grid"], cfg["eos"], cfg["kin"], k, transport=transport)
    many.init(cfg["init"])
    if case == "periodic-x":                    # give the periodic box something to do: a pressure pulse through init_fields
        q = one.state()
        q[4][:, :6] *= 40.0                     # ... that crosses the wrap-around seam in both directions
        q[4][:, -5:] *= 40.0
        one.init_fields(q)
        for s, (x0, n) in zip(many.sims, many.parts):
            s.init_fields([a[:, x0:x0 + n] for a in q])
    for a, b in zip(one.state(), many.state()):
        assert np.array_equal(a, b)             # sim_init_slab paints the slab's columns of the same field
    one.step(steps)
    many.step(steps)
    for f, (a, b) in enumerate(zip(one.state(), many.state())):
        assert np.array_equal(a, b), "plane %d differs, max |diff| %g" % (f, np.abs(a - b).max())
    d1, dk = one.diagnostics(), many.diagnostics()
    assert d1["t"] == dk["t"] and d1["step"] == dk["step"] == steps and d1["dt_last"] == dk["dt_last"]
    for key in ("M2r", "M2tot0", "mass1", "mass2", "momx", "energy"):
        assert dk[key] == pytest.approx(d1[key], rel=1e-12, abs=1e-9 * abs(d1["mass2"]))
    assert dk["smax"] == d1["smax"] and dk["bad_state"] == 0
    one.close(), many.close()


def test_local_slabs_fixed_dt_then_cfl_and_resume(B):
    """fixed-dt steps, then CFL-limited ones, then more after reading the state back (the driver re-enters cleanly)"""
    from paper_1905_05727_b200 import slab
    cfg = inputs.config("C1")
    one = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    one.init(cfg["init"])
    many = slab.LocalSlabs(cfg["grid"], cfg["eos"], cfg["kin"], 2, transport="peer")
    many.init(cfg["init"])
    dt = 0.5 * one.cfl_dt()
    one.step_dt(7, dt), many.step(7, dt_fixed=dt)
    one.step(8), many.step(8)
    assert all(np.array_equal(a, b) for a, b in zip(one.state(), many.state()))
    one.step(5), many.step(5)
    assert all(np.array_equal(a, b) for a, b in zip(one.state(), many.state()))
    assert one.diagnostics()["t"] == many.diagnostics()["t"]


def test_decomposed_step_against_the_oracle(O, B):
    """the parity gate itself on the decomposed path: 3 slabs, 1 step and 20 steps of C1 against the oracle"""
    from paper_1905_05727_b200 import slab
    cfg = inputs.config("C1")
    o = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=8)
    o.init(cfg["init"])
    for _ in range(150):                         # bring the shock into the cavity with the oracle alone
        o.step(1)
    q0 = o.state()
    many = slab.LocalSlabs(cfg["grid"], cfg["eos"], cfg["kin"], 3, transport="peer")
    many.init(cfg["init"])
    for s, (x0, n) in zip(many.sims, many.parts):
        s.init_fields([a[:, x0:x0 + n] for a in q0])
    many._begun = None
    t0 = o.diagnostics()["t"]                    # init_fields restarts the slabs' clock at 0
    dt = o.cfl_dt()
    o.step_dt(1, dt), many.step(1, dt_fixed=dt)
    r = rel_diff(many.state(), o.state(), o.read_field("c"))
    assert max(r) <= TOL_ONE_STEP, r
    o.step(20), many.step(20)
    r = l1_rel(many.state(), o.state())
    assert max(r) <= 1e-9, r
    assert many.diagnostics()["t"] == pytest.approx(o.diagnostics()["t"] - t0, rel=1e-10)


def test_slab_argument_checks(B):
    cfg = inputs.config("C1", nx=64, ny=32)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    with pytest.raises(B.NmsdtError) as e:
        s.slab_pass(1)                                                   # not initialised
    assert e.value.code == B.SIM_ERR_STATE
    s.init(cfg["init"])
    assert s.slab_halo_bytes() == 7 * 32 * 2 * 8
    with pytest.raises(B.NmsdtError) as e:
        s.slab_pass(3)
    assert e.value.code == B.SIM_ERR_ARG
    info = s.slab_info()
    assert info.nx == 64 and info.ny == 32 and info.plane0[0] and info.plane0[1]
    bad = B.SlabPeer()
    bad.plane0[0], bad.plane0[1], bad.plane_stride, bad.pitch, bad.nx, bad.ny = info.plane0[0], info.plane0[1], info.plane_stride, info.pitch, 64, 31
    with pytest.raises(B.NmsdtError) as e:
        s.slab_connect(0, bad)                                           # neighbour with another ny
    assert e.value.code == B.SIM_ERR_ARG
    with pytest.raises(B.NmsdtError) as e:
        s.slab_ipc_export()                                              # workspace lent by torch: no IPC export
    assert e.value.code == B.SIM_ERR_STATE
    s.set_variant(B.VARIANT_UNFUSED)
    with pytest.raises(B.NmsdtError) as e:
        s.slab_pass(1)
    assert e.value.code == B.SIM_ERR_STATE
    g = dict(cfg["grid"], bc_ylo=4, bc_yhi=4)                            # EXTERNAL is an x-side kind only
    with pytest.raises(B.NmsdtError):
        B.Sim(g, cfg["eos"], cfg["kin"])
    own = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], library_workspace=True)
    own.init(cfg["init"])
    handle, oa, ob = own.slab_ipc_export()
    assert len(handle) == 64 and ob > oa >= 0


WORKER = r"""
import os, sys
sys.path.insert(0, %(root)r)
import numpy as np, torch, torch.distributed as dist
from paper_1905_05727_b200 import binding, inputs, slab
torch.cuda.set_device(0)
dist.init_process_group("gloo")
rank = dist.get_rank()
out, transport = sys.argv[1], sys.argv[2]
cfg = inputs.config("C4", nx=512, ny=128)
mk = lambda g: binding.Sim(g, cfg["eos"], cfg["kin"], library_workspace=(transport == "peer"))
ds = slab.DistSlab(cfg["grid"], mk, dist, "cuda:0", transport=transport)
ds.init(cfg["init"])
ds.step(12)
d = ds.diagnostics()
np.savez(os.path.join(out, "%%s_rank%%d.npz" %% (transport, rank)), q=np.stack(ds.sim.state()), t=d["t"], M2r=d["M2r"], x0=ds.x0)
dist.barrier()
ds.close()
dist.destroy_process_group()
"""


@pytest.mark.parametrize("transport,port", [("staged", 29631), ("peer", 29632)])
def test_distslab_two_processes_on_one_gpu(B, tmp_path, transport, port):
    w = tmp_path / "worker.py"
    w.write_text(WORKER % dict(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                        "127.0.0.1", "--master-port", str(port), str(w), str(tmp_path), transport],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=900)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    cfg = inputs.config("C4", nx=512, ny=128)
    one = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    one.init(cfg["init"])
    one.step(12)
    parts = [np.load(tmp_path / ("%s_rank%d.npz" % (transport, rk))) for rk in range(2)]
    q = np.concatenate([p["q"] for p in parts], axis=2)
    assert np.array_equal(q, np.stack(one.state()))
    d = one.diagnostics()
    for p in parts:
        assert float(p["t"]) == d["t"] and float(p["M2r"]) == pytest.approx(d["M2r"], rel=1e-12)


@pytest.mark.parametrize("transport,port", [("staged", 29641), ("peer", 29642)])
def test_bench_decomp_slab_two_ranks_on_one_gpu(B, transport, port):
    """`bench.py --decomp slab` under torchrun, as the driver would launch it for N = 2, on the one GPU there is (the ranks
    share it and gloo carries the collectives: a plumbing check, not a measurement): one JSON line from rank 0, a domain of
    2 x C3's columns advanced by both ranks to the same step, finite state."""
    import json
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                        "127.0.0.1", "--master-port", str(port), "bench.py", "--gpus", "2", "--steps", "4", "--warmup", "3",
                        "--config", "C3", "--decomp", "slab", "--transport", transport],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=900)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["config"]["parallelism"] == "x-slabs" and d["config"]["ranks_share_a_gpu"] is True
    assert d["sim"]["step"] == 7 and d["sim"]["bad_state"] == 0 and d["value"] > 0 and d["gpu_launches"] > 0
    # the same domain undivided, same number of steps: identical clock and (up to summation order) identical reactive mass
    cfg = inputs.config("C3")
    g = dict(cfg["grid"], nx=2 * cfg["grid"]["nx"])
    ini = dict(cfg["init"], x_hi=g["nx"])
    one = B.Sim(g, cfg["eos"], cfg["kin"])
    one.init(ini)
    one.step(7)
    d1 = one.diagnostics()
    assert d["sim"]["t"] == d1["t"] and d["sim"]["M2r"] == pytest.approx(d1["M2r"], rel=1e-12)
