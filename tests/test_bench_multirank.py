"""N > 1 launch of bench.py on CPU (gloo, world_size 2): the path does not shard (replicas only),
so the multi-rank logic is the max-over-ranks timing, the whole-job aggregate, and the reference arm's rule that rank 0
alone runs and prints."""
import json
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")          # rank 1 is the slow one
v = bench.aggregate_value(1000, 4, world, ms * 1e-3)
print("RESULT %%d %%r %%r" %% (rank, ms, v), flush=True)
dist.destroy_process_group()
"""


def _torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    return subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args,
                          capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)


def test_max_over_ranks_and_aggregate_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER % ROOT)
    r = _torchrun([str(w)], 29611)
    assert r.returncode == 0, r.stderr[-2000:]
    res = re.findall(r"RESULT (\d) ([0-9.e+-]+?) ([0-9.e+-]+?)(?=RESULT|\s|$)", r.stdout)    # the two ranks' lines may interleave
    assert sorted(x[0] for x in res) == ["0", "1"]
    for rank, ms, v in res:
        assert float(ms) == 15.0                                   # the slowest rank's time on every rank
        assert float(v) == 1000 * 4 * 2 / 15e-3                    # units of both replicas / max time


def test_reference_arm_under_torchrun_prints_once():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "C1"], 29612)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0
