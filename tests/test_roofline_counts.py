"""The roofline block of bench.py is computed from ncu counts of the sweep kernels (profiles/roofline_counts.json).  The file
carries a hash of the kernel sources: these tests fail when a kernel source was edited and the counts were not taken again
(`python roofline_counts.py`, see its docstring), so `roofline.frac` cannot silently drift from the build."""
import json
import os

import roofline_counts

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _counts():
    with open(os.path.join(ROOT, "profiles", "roofline_counts.json")) as f:
        return json.load(f)


def test_counts_belong_to_the_kernel_sources_in_the_tree():
    c = _counts()
    assert c["source_sha256"] == roofline_counts.source_hash(), (
        "kernel sources changed since the ncu capture behind profiles/roofline_counts.json: capture again and rerun "
        "python roofline_counts.py")
    assert c["source_files"] == ["paper_1905_05727_b200/" + f for f in roofline_counts.SOURCES]
    assert c["ncu_command"].startswith("ncu ") and "bench.py" in c["ncu_command"]


def test_counts_are_complete_and_plausible():
    k = _counts()["kernels"]
    assert sorted(k) == ["x_lead", "x_trail", "y_lead", "y_trail"]
    for name, v in k.items():
        # a fused sweep executes a few hundred FP64-pipe instructions per cell, about as many others, and moves the 7 planes once each way
        assert 250 < v["fp64_instr_per_cell"] < 500 and v["fp64_instr_per_cell"] < v["warp_instr_per_cell"] < 1000, name
        assert 111.9 < v["dram_bytes_per_cell"] < 118.0, name                      # 112 B algorithmic
        assert abs(v["flop_per_cell"] - (2 * v["dfma_dmul_dadd_per_cell"][0] + sum(v["dfma_dmul_dadd_per_cell"][1:]))) < 1e-6
        assert 1.0 < v["executed_over_algorithmic"] < 1.1
    assert k["x_trail"]["fp64_instr_per_cell"] > k["x_lead"]["fp64_instr_per_cell"]      # pass 2 carries the wavespeed and the state check


def test_bench_reads_the_counts_and_flags_stale_ones(tmp_path, monkeypatch):
    import importlib.util
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    c, stale = bench.load_counts()
    assert stale is False and c["kernels"]["y_trail"]["fp64_instr_per_cell"] > 0
    monkeypatch.setattr(roofline_counts, "source_hash", lambda: "0" * 64)
    assert bench.load_counts()[1] is True
