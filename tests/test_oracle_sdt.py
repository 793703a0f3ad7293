"""End-to-end soft pin of the whole oracle step (O1-O8) against the numbers the paper prints for neat NM at
7.81 GPa: overtake time 4.22 us (their dx = 1 um; here dx = 16 um, grid-converged to 0.3 %),
negligible global reaction rate before 2.4 us, rapid rise at 2.6-2.8 us, abrupt peak and drop at overtake.
The 3 % offset to 4.22 us is the unknown wave-speed / CFL / boundary detail of the paper's code."""
import os

import numpy as np
import pytest

from paper_1905_05727_b200 import inputs


def _golden():
    vals = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = float(v)
    return vals


@pytest.mark.slow
def test_neat_nm_overtake_time_and_rate_curve(O):
    g = _golden()
    dx, L, Ls = 16e-6, 24e-3, 0.5e-3
    nx, sc = int(round((L + Ls) / dx)), int(round(Ls / dx))
    grid = dict(nx=nx, ny=1, dx=dx, dy=dx, bc_xlo=0, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)
    init = dict(inputs._INIT0, p_shock=7.81e9, shock_cells=sc)
    o = O.Oracle(grid, inputs.EOS, inputs.KIN)
    o.init(init)
    ts, Ms = [0.0], [o.diagnostics()["M2r"]]
    while ts[-1] < 4.7e-6:
        o.step(10)                      # R14: sample every 10 steps, backward difference
        d = o.diagnostics()
        ts.append(d["t"])
        Ms.append(d["M2r"])
    assert d["bad_state"] == 0 and o.fallback_count() == 0
    ts, Ms = np.array(ts), np.array(Ms)
    rate = np.abs(np.diff(Ms)) / np.diff(ts) / d["M2tot0"]     # Eq. 13
    tm = 0.5 * (ts[1:] + ts[:-1])
    k = int(np.argmax(rate))
    t_ov = tm[k]
    assert t_ov == pytest.approx(g["overtake_neat_us"] * 1e-6, rel=0.05)
    at = lambda t_us: rate[np.argmin(np.abs(tm - t_us * 1e-6))]
    assert np.all(rate[tm < g["rate_quiet_until_us"] * 1e-6] < 0.05 * rate[k])     # "insignificant before 2.4 us"
    assert at(2.8) > 3.0 * at(2.6)                                                  # "rapid increase at 2.6-2.8 us"
    assert at(4.0) < 1.25 * at(3.2)                                                 # "slows down after 3.2 us"
    assert at(t_ov * 1e6 + 0.3) < 0.5 * rate[k]                                     # "abrupt decrease" after the peak
    assert 5e5 < rate[k] < 2e6
    # superdetonation: pressure behind the overtaking wave far above the 7.81 GPa input and above CJ
    assert o.read_field("p").max() > 15e9
