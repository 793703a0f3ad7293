"""Turn an ncu capture of the four fused sweep kernels into the per-cell counts that bench.py's `roofline` block uses,
tied to the kernel sources by a hash (profiles/roofline_counts.json).

    # on the GPU box (after the same bench command has exited 0 without ncu; B200_PROFILING.md):
    ncu --set full --metrics sm__inst_executed_pipe_fp64.sum,smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,\
smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,smsp__sass_thread_inst_executed_op_dadd_pred_on.sum \
        --clock-control none --import-source on -k regex:k_[xy]sweep -s 6 -c 4 -o gpurun_out/sweeps_c5 -f \
        python bench.py --steps 2 --warmup 3 --no-e2e --no-cpu --no-slab
    # here (no GPU needed):
    ncu -i gpurun_out/sweeps_c5.ncu-rep --page raw --csv > sweeps_c5_raw.csv
    python roofline_counts.py sweeps_c5_raw.csv --nx 32768 --ny 4096 --seg-x 3644 --seg-y 256 \
        --command "<the ncu command>" --out profiles/roofline_counts.json

What is counted: warp instructions executed on the FP64 pipe (DADD, DMUL, DFMA, DSETP alike: each holds
the half-rate pipe -- and the scheduler's issue port -- for two cycles), all warp instructions, thread-level DFMA / DMUL / DADD
for the plain flop count, DRAM bytes.  "Per cell" = per cell of the grid per launch; the kernels execute (seg + ramp)/seg times
the algorithmic work (ramp-up cells of every segment, `sim_sweep_geometry`), which is divided out.
"""
import argparse
import csv
import hashlib
import json
import os
import re

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_1905_05727_b200")
# everything the sweep kernels are compiled from: a change to any of these files invalidates the counts
SOURCES = ["csrc/nmsdt_fused.cu", "csrc/nmsdt_fast.cuh", "csrc/nmsdt_math.cuh", "csrc/nmsdt_device.cuh"]
MODES = {1: "lead", 2: "trail", 0: "plain", 3: "trail_inert"}
N_SM = 148


def source_hash():
    h = hashlib.sha256()
    for f in SOURCES:
        with open(os.path.join(HERE, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _num(x):
    try:
        return float(x.replace(",", ""))
    except ValueError:
        return None


def parse(raw_csv):
    rows = list(csv.reader(open(raw_csv)))
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "msecond": 1e-3, "usecond": 1e-6, "second": 1.0, "ms": 1e-3, "us": 1e-6,
             "ns": 1e-9, "nsecond": 1e-9}

    def get(r, name, default=None):
        if name not in col:
            return default
        v = _num(r[col[name]])
        if v is None:
            return default
        return v * scale.get(units[col[name]], 1.0)

    out = []
    for r in rows[2:]:
        name = r[col["Kernel Name"]]
        m = re.search(r"k_([xy])sweep<\(?(?:int\))?(\d)\s*,\s*\(?(?:int\))?(\d)>", name)
        if not m:
            continue
        cyc = get(r, "sm__cycles_active.avg")
        fp64 = get(r, "sm__inst_executed_pipe_fp64.sum")
        pct = get(r, "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active")
        if fp64 is None:        # capture without the explicit metric: 2 warp instructions per cycle and SM at 100 %
            fp64 = pct / 100.0 * cyc * 2.0 * N_SM
        el = get(r, "sm__cycles_elapsed.avg", cyc)

        def thread_op(op):
            v = get(r, "smsp__sass_thread_inst_executed_op_%s_pred_on.sum" % op)
            if v is None:
                v = get(r, "smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % op) * el
            return v

        out.append({"dir": m.group(1), "mode": MODES[int(m.group(2))], "limiter": int(m.group(3)),
                    "ms": get(r, "gpu__time_duration.sum") * 1e3, "fp64_warp_instr": fp64, "warp_instr": get(r, "smsp__inst_executed.sum"),
                    "dfma": thread_op("dfma"), "dmul": thread_op("dmul"), "dadd": thread_op("dadd"),
                    "dram_bytes": get(r, "dram__bytes_read.sum") + get(r, "dram__bytes_write.sum"),
                    "fp64_pipe_pct": pct, "issue_active_pct": get(r, "smsp__issue_active.avg.pct_of_peak_sustained_active"),
                    "registers": get(r, "launch__registers_per_thread"), "grid": get(r, "launch__grid_size")})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--nx", type=int, required=True)
    ap.add_argument("--ny", type=int, required=True)
    ap.add_argument("--seg-x", type=int, required=True, help="sim_sweep_geometry(0): segment length (bench.py prints it)")
    ap.add_argument("--seg-y", type=int, required=True)
    ap.add_argument("--ramp-x", type=int, default=4)
    ap.add_argument("--ramp-y", type=int, default=4)
    ap.add_argument("--workload", default="C5")
    ap.add_argument("--command", default="", help="the ncu command that made the capture")
    ap.add_argument("--round", default="r02")
    ap.add_argument("--out", default=os.path.join(HERE, "..", "profiles", "roofline_counts.json"))
    a = ap.parse_args()
    cells = float(a.nx) * a.ny
    red = {"x": (a.seg_x + a.ramp_x) / a.seg_x, "y": (a.seg_y + a.ramp_y) / a.seg_y}
    ks = {}
    for k in parse(a.raw_csv):
        key = "%s_%s" % (k["dir"], k["mode"])
        r = red[k["dir"]]
        ks[key] = {"ms_under_ncu": k["ms"], "registers": k["registers"], "grid_blocks": k["grid"], "fp64_pipe_pct": k["fp64_pipe_pct"],
                   "issue_active_pct": k["issue_active_pct"],
                   "fp64_instr_per_cell": k["fp64_warp_instr"] * 32.0 / cells / r,
                   "warp_instr_per_cell": k["warp_instr"] * 32.0 / cells / r,
                   "flop_per_cell": (2.0 * k["dfma"] + k["dmul"] + k["dadd"]) / cells / r,
                   "dfma_dmul_dadd_per_cell": [k["dfma"] / cells / r, k["dmul"] / cells / r, k["dadd"] / cells / r],
                   "dram_bytes_per_cell": k["dram_bytes"] / cells, "executed_over_algorithmic": r}
    out = {"round": a.round, "workload": "%s %dx%d" % (a.workload, a.nx, a.ny), "geometry": {"seg_x": a.seg_x, "ramp_x": a.ramp_x, "seg_y": a.seg_y, "ramp_y": a.ramp_y},
           "source_sha256": source_hash(), "source_files": ["paper_1905_05727_b200/" + f for f in SOURCES], "ncu_command": a.command,
           "counting": "per cell of the grid and launch; FP64-pipe and all warp instructions x 32 / cells / ((seg + ramp)/seg); "
                       "flops: dfma = 2, dmul = dadd = 1, dsetp = 0 (thread level, predicated on)",
           "kernels": ks}
    with open(a.out, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")
    for key in sorted(ks):
        print("%-8s FP64 %.1f  all %.1f  flop %.1f  DRAM %.1f B/cell  (%.3f ms under ncu, FP64 pipe %.1f %%)" % (
            key, ks[key]["fp64_instr_per_cell"], ks[key]["warp_instr_per_cell"], ks[key]["flop_per_cell"], ks[key]["dram_bytes_per_cell"],
            ks[key]["ms_under_ncu"], ks[key]["fp64_pipe_pct"]))


if __name__ == "__main__":
    main()
