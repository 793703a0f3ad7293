"""Paper-scale validation runs: the paper's three scenarios at its own domain sizes, run through
the C ABI on one GPU, reporting the detonation overtake time = time of the peak of the normalised global reaction rate
(Eq. 12-13).

    python -m paper_1905_05727_b200.validate --case neat|regular|random [--dx 1] [--phi 0.08] [--t-end 4.8e-6]

What the paper prints for d_c = 100 um, 7.81 GPa (other machine, its own unknown numerical details; context, not a pin of
this code): neat 4.22 us; regular phi = 8 %: 3.77 / 3.05 / 2.88 / 2.88 us at dx = 4 / 2 / 1 / 0.5 um (Table IV);
random phi = 5 %: 3.68 / 3.21 / 2.99 us at dx = 4 / 2 / 1 um (Table V); random phi = 8 %: 2.67 us at dx = 1 um.
Only argument marshalling and the bookkeeping of the sampled curve happen here; every step runs in the kernels.
"""
import argparse
import json
import time

import numpy as np

from . import binding, inputs

PAPER_US = {("neat", 1.0, None): 4.22,
            ("regular", 4.0, 0.08): 3.77, ("regular", 2.0, 0.08): 3.05, ("regular", 1.0, 0.08): 2.88, ("regular", 0.5, 0.08): 2.88,
            ("random", 4.0, 0.05): 3.68, ("random", 2.0, 0.05): 3.21, ("random", 1.0, 0.05): 2.99, ("random", 1.0, 0.08): 2.67}


def run(case, dx_um=1.0, phi=None, t_end=None, sample_every=10, seed=2019, verbose=False, p_shock=7.81e9, length_mm=24.0,
        limiter=None, samples=False):
    """One validation run.  p_shock / length_mm / limiter (inputs.LIM_MINMOD, inputs.LIM_MC; R5) default to the
    paper's case and this build's default limiter; samples=True adds the full sampled curve ("t", "M2r") to the result."""
    cfg = inputs.paper_case(case, dx_um, p_shock=p_shock, phi=phi, seed=seed, length_mm=length_mm)
    g, ini = cfg["grid"], cfg["init"]
    if limiter is not None:
        g["limiter"] = int(limiter)
    if t_end is None:
        t_end = 4.8e-6 if case == "neat" else 4.4e-6
    sim = binding.Sim(g, cfg["eos"], cfg["kin"])
    t0 = time.perf_counter()
    sim.init(ini)
    d = sim.diagnostics()
    ts, M = [0.0], [d["M2r"]]
    xt, xs = [0.0], [ini["shock_cells"] * g["dx"]]
    steps = 0
    x_stop = (g["nx"] - 64) * g["dx"]
    while d["t"] < t_end:
        sim.step(sample_every)
        steps += sample_every
        d = sim.diagnostics()
        ts.append(d["t"]); M.append(d["M2r"])
        if steps % (10 * sample_every) == 0:
            x = sim.profiles(1.01 * ini["p0"])[3]
            xt.append(d["t"]); xs.append(x)
            if x >= x_stop:
                break
    wall = time.perf_counter() - t0
    ts, M = np.array(ts), np.array(M)
    rate = np.abs(np.diff(M)) / np.diff(ts) / d["M2tot0"]          # R14: backward differences, assigned to the mid time
    tm = 0.5 * (ts[1:] + ts[:-1])
    k = int(np.argmax(rate))
    # Appendix C: time of the maximum shock acceleration (Eq. C1-C2 with the paper's 1.5 us window, where it fits)
    t_amax = None
    xt, xs = np.array(xt), np.array(xs)
    if xt[-1] - xt[0] > 3.2e-6:
        _, acc = sim.shock_kinematics(xt, xs, 1.5e-6)
        valid = np.flatnonzero(~np.isnan(acc))
        if valid.size > 2:
            ka = int(np.nanargmax(acc))
            if valid[0] < ka < valid[-1]:          # a maximum at the edge of the window is not a maximum
                t_amax = float(xt[ka])
    cav = sim.cavities() if case != "neat" else np.zeros((0, 3))
    ncav = len(cav)
    # air fraction actually placed (a generator that ran out of candidates used to return a thinner field silently;
    # sim_init now fails in that case, and the achieved value is reported either way)
    phi_placed = float(np.pi * np.sum(cav[:, 2] ** 2) / ((g["nx"] - ini["shock_cells"]) * g["ny"])) if ncav else 0.0
    sim.close()
    key = (case, float(dx_um), None if case == "neat" else (phi if phi is not None else (0.08 if case == "regular" else 0.05)))
    out = {"case": cfg["name"], "grid": [g["nx"], g["ny"]], "dx_um": dx_um, "phi": key[2], "phi_placed": phi_placed, "cavities": ncav,
           "limiter": "MC" if g["limiter"] == inputs.LIM_MC else "minmod", "p_shock": p_shock, "steps": steps,
           "t_final_us": float(d["t"]) * 1e6, "overtake_us": float(tm[k]) * 1e6, "peak_rate_per_s": float(rate[k]),
           "t_max_shock_acceleration_us": None if t_amax is None else t_amax * 1e6,
           "paper_overtake_us": PAPER_US.get(key) if (p_shock == 7.81e9 and length_mm == 24.0) else None, "bad_state": int(d["bad_state"]), "wall_s": wall,
           "gcell_updates_per_s": g["nx"] * g["ny"] * steps / wall / 1e9}
    if samples:
        out["t"], out["M2r"], out["M2tot0"] = ts, M, float(d["M2tot0"])
    if verbose:
        out["curve_t_us"] = (tm[::20] * 1e6).round(4).tolist()
        out["curve_rate"] = rate[::20].tolist()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--case", default="neat", choices=["neat", "regular", "random"])
    ap.add_argument("--dx", type=float, default=1.0, help="grid spacing in um (paper: 1)")
    ap.add_argument("--phi", type=float, default=None)
    ap.add_argument("--t-end", type=float, default=None)
    ap.add_argument("--seed", type=int, default=2019)
    ap.add_argument("--curve", action="store_true")
    ap.add_argument("--limiter", default=None, choices=["minmod", "mc"], help="slope limiter (DESIGN.md R5); default: the build's default")
    ap.add_argument("--p-shock", type=float, default=7.81e9)
    ap.add_argument("--length-mm", type=float, default=24.0)
    a = ap.parse_args()
    lim = None if a.limiter is None else (inputs.LIM_MC if a.limiter == "mc" else inputs.LIM_MINMOD)
    print(json.dumps(run(a.case, a.dx, a.phi, a.t_end, seed=a.seed, verbose=a.curve, p_shock=a.p_shock, length_mm=a.length_mm, limiter=lim)))


if __name__ == "__main__":
    main()
