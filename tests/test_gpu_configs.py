"""GPU parity on BASELINE.json's five configs at their own sizes (SURVEY.md 8(d) "Parity workload"), at north_star's three
tolerances: max relative difference per conserved variable <= 1e-11 after one step, L1-relative <= 1e-7 after 500 steps,
global-reaction-rate curve (Eq. 12-13) and overtake time within 0.5 %.

  C1  256 x 128, 200 steps (+ 500)                       tests/test_gpu_parity.py
  C2  4096 x 32 at 8, 9.4 and 11 GPa, each run until the global reaction rate has peaked       here
  C3  4096 x 512, 500 steps                               here
  C4  8192 x 1024: here the full grid for 500 steps at 8 GPa; a 2048 x 512 crop at each of the config's three input
      pressures (7, 8, 9 GPa); a 1024 x 256 crop at 9 GPa through cavity collapse and hot-spot ignition with diagnostics
      every 10 steps (1 step on the full grid on sampled windows: tests/test_gpu_parity.py)
  C5  32768 x 4096: 1 step on the full grid in tests/test_gpu_parity.py; here the 4096 x 1024 crop SURVEY 8(d) names
      (6.7e10 oracle cell-updates for the full grid are out of reach), 500 steps

Both sides start from the oracle's initial state and then keep their own state (no re-synchronisation): the GPU takes
its own device-side CFL step.  One-step parity on developed states is checked on a second handle that is handed the
oracle's state at that moment.  The oracle runs on all host cores (OpenMP over rows, bit-identical to one thread).
"""
import os

import numpy as np
import pytest

from paper_1905_05727_b200 import inputs
from parity_util import TOL_L1_500, TOL_ONE_STEP, TOL_RATE, l1_rel, rate_curve, rel_diff

pytestmark = pytest.mark.gpu
THREADS = os.cpu_count() or 1


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1905_05727_b200 import binding, build
    build.build()
    binding.load_library()
    return binding


def _start(O, B, cfg, variant=1):
    """oracle and GPU handle on the same initial state (the oracle's)"""
    o = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=THREADS)
    o.init(cfg["init"])
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant)
    s.init_fields(o.state())
    return o, s


def _one_step_from(O, B, cfg, o, what, variants=(1,)):
    """hand the oracle's current state to fresh handles and compare one even and one odd step"""
    q = o.state()
    o2 = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=THREADS)
    o2.init_fields(q)
    sims = [B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=v) for v in variants]
    for s2 in sims:
        s2.init_fields(q)
    for it in range(2):
        o2.step(1)
        c = o2.read_field("c")
        for v, s2 in zip(variants, sims):
            s2.step(1)
            r = rel_diff(s2.state(), o2.state(), c)
            assert max(r) <= (it + 1) * TOL_ONE_STEP, "%s variant %d step %d: %s" % (what, v, it, r)
    assert o2.fallback_count() == 0
    for s2 in sims:
        s2.close()


def _assert_curves(ta, Ma, M0a, tb, Mb, M0b, what, need_peak=True):
    """Eq. 13 by backward differences of the samples (R14): curve within 0.5 % wherever the rate exceeds 1 % of its peak,
    overtake time (time of the peak) within 0.5 %"""
    tma, ra = rate_curve(ta, Ma, M0a)
    tmb, rb = rate_curve(tb, Mb, M0b)
    k = int(np.argmax(rb))
    if need_peak:
        assert 5 < k < len(rb) - 5, "%s: the rate peak must lie inside the run (k = %d of %d)" % (what, k, len(rb))
    sig = rb > 0.01 * rb[k]
    assert sig.sum() >= 10, what
    dev = float(np.max(np.abs(ra[sig] / rb[sig] - 1.0)))
    assert dev < TOL_RATE, "%s: rate curve deviates by %.3g" % (what, dev)
    assert tma[int(np.argmax(ra))] == pytest.approx(tmb[k], rel=TOL_RATE), what
    np.testing.assert_allclose(ta, tb, rtol=1e-9)
    return tmb[k], rb[k], dev


# ------------------------------------------------------------------------------------------------ C2
@pytest.mark.slow
@pytest.mark.parametrize("p_gpa", [11.0, 9.4, 8.0])
def test_c2_full_strip_until_the_rate_has_peaked(O, B, p_gpa):
    """BASELINE config 2 at its real size: neat NM, 4096 x 32, dx = 5 um, run until the global reaction rate has peaked
    (thermal explosion -> superdetonation -> overtake); samples every 10 steps"""
    cfg = inputs.config("C2", p_shock=p_gpa * 1e9)
    o, s = _start(O, B, cfg)
    _one_step_from(O, B, cfg, o, "C2 %g GPa initial state" % p_gpa, variants=(0, 1))
    ta, Ma, tb, Mb = [0.0], [s.diagnostics()["M2r"]], [0.0], [o.diagnostics()["M2r"]]
    M0 = o.diagnostics()["M2tot0"]
    best, since, n, cap = 0.0, 0, 0, 30000
    checked_mid = False
    while True:
        o.step(10), s.step(10)
        n += 10
        da, db = s.diagnostics(), o.diagnostics()
        ta.append(da["t"]); Ma.append(da["M2r"]); tb.append(db["t"]); Mb.append(db["M2r"])
        if n == 500:
            l1 = l1_rel(s.state(), o.state())
            assert max(l1) <= TOL_L1_500, "C2 %g GPa, 500 steps: %s" % (p_gpa, l1)
        r = abs(Mb[-1] - Mb[-2]) / (tb[-1] - tb[-2]) / M0
        if r > best:
            best, since = r, 0
        else:
            since += 1
        if not checked_mid and best > 2e4 and r > 0.5 * best:           # the reaction wave is running: developed state
            _one_step_from(O, B, cfg, o, "C2 %g GPa at step %d" % (p_gpa, n))
            checked_mid = True
        if (since >= 30 and best > 1e4) or n >= cap:
            break
    assert n < cap and checked_mid and da["bad_state"] == 0 and da["step"] == db["step"] == n
    t_ov, peak, dev = _assert_curves(np.array(ta), np.array(Ma), da["M2tot0"], np.array(tb), np.array(Mb), M0, "C2 %g GPa" % p_gpa)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= 100 * TOL_L1_500, l1          # after thousands of steps through a detonation: still tiny
    assert db["burned_mass"] > 0.05 * M0
    # the physics the run must show: higher input pressure, earlier overtake; ~3.5 / 1.1 / 0.4 us
    lo, hi = {11.0: (0.2e-6, 0.7e-6), 9.4: (0.6e-6, 1.8e-6), 8.0: (2.0e-6, 4.5e-6)}[p_gpa]
    assert lo < t_ov < hi, t_ov
    print("C2 %g GPa: %d steps, overtake %.4f us, peak rate %.3e /s, curve deviation %.2e, final L1 %.2e" % (p_gpa, n, t_ov * 1e6, peak, dev, max(l1)))


# ------------------------------------------------------------------------------------------------ C3
@pytest.mark.slow
def test_c3_full_regular_array_500_steps(O, B):
    """BASELINE config 3 at its real size, 4096 x 512, 448 lattice cavities, 8 GPa: one step and 500 steps"""
    cfg = inputs.config("C3")
    o, s = _start(O, B, cfg)
    assert len(o.cavities()) == 448
    o.step(1), s.step(1)
    r = rel_diff(s.state(), o.state(), o.read_field("c"))
    assert max(r) <= TOL_ONE_STEP, r
    o.step(499), s.step(499)
    da, db = s.diagnostics(), o.diagnostics()
    assert da["step"] == db["step"] == 500 and da["bad_state"] == 0
    assert da["t"] == pytest.approx(db["t"], rel=1e-10)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= TOL_L1_500, l1
    for k in ("M2r", "mass1", "mass2", "momx", "energy"):
        assert da[k] == pytest.approx(db[k], rel=1e-11), k
    assert o.fallback_count() == 0
    print("C3 full, 500 steps: L1 %s" % (["%.1e" % v for v in l1],))


# ------------------------------------------------------------------------------------------------ C4
@pytest.mark.slow
def test_c4_crop_cavity_collapse_rate_curve(O, B):
    """The hot-spot-driven reaction rate: a 1024 x 256 crop of BASELINE config 4 (random cavities d = 24,
    gap 4, phi = 3 %, seed 12345) at its highest input pressure, 9 GPa, diagnostics every 10 steps through collapse and
    ignition of the first cavities; 500-step L1 on the way, one-step parity on the developed state at the end"""
    cfg = inputs.config("C4", nx=1024, ny=256, p_shock=9e9)
    o, s = _start(O, B, cfg)
    cav = o.cavities()
    assert len(cav) >= 10
    ta, Ma, tb, Mb = [0.0], [s.diagnostics()["M2r"]], [0.0], [o.diagnostics()["M2r"]]
    nsteps = 1800
    for n in range(10, nsteps + 1, 10):
        o.step(10), s.step(10)
        da, db = s.diagnostics(), o.diagnostics()
        ta.append(da["t"]); Ma.append(da["M2r"]); tb.append(db["t"]); Mb.append(db["M2r"])
        if n == 500:
            l1 = l1_rel(s.state(), o.state())
            assert max(l1) <= TOL_L1_500, l1
    M0 = db["M2tot0"]
    tb_, Mb_ = np.array(tb), np.array(Mb)
    _, rb = rate_curve(tb_, Mb_, M0)
    # the shock (about 0.3 cells per step) has crossed the first cavities: their collapse ignites the liquid around them and the
    # global rate rises several times over the induction-time rate of the shocked neat liquid
    x_first = cav[:, 0].min()
    k_before = max(2, int((x_first - cav[:, 2].max() - 120) / 0.45 / 10) - 5)
    assert rb[-1] > 5 * rb[k_before], (rb[k_before], rb[-1])
    _assert_curves(np.array(ta), np.array(Ma), da["M2tot0"], tb_, Mb_, M0, "C4 crop", need_peak=False)
    assert da["bad_state"] == 0 and o.fallback_count() == 0
    T2 = o.read_field("T2")
    assert T2.max() > 1600.0            # hot spots well above the ~1064 K of the 9 GPa shock
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= 10 * TOL_L1_500, l1
    _one_step_from(O, B, cfg, o, "C4 crop after %d steps" % nsteps, variants=(0, 1))
    print("C4 crop: rate %.3e -> %.3e /s, final L1 %.2e, T2max %.0f K" % (rb[k_before], rb[-1], max(l1), T2.max()))


@pytest.mark.parametrize("p_shock", [7e9, 8e9, 9e9])
def test_c4_one_step_and_early_run_at_each_input_pressure(O, B, p_shock):
    """BASELINE config 4's three input shock pressures, 7 / 8 / 9 GPa (the random-cavity rate curves), on a
    2048 x 512 crop with the config's generator parameters: one step on the initial state (both variants), 60 steps of
    free running (own device-side CFL steps), one even and one odd step on the developed state"""
    cfg = inputs.config("C4", nx=2048, ny=512, p_shock=p_shock)
    o, s = _start(O, B, cfg)
    assert len(o.cavities()) > 20
    s0 = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=0)
    s0.init_fields(o.state())
    o.step(1), s.step(1), s0.step(1)
    c = o.read_field("c")
    for h in (s, s0):
        r = rel_diff(h.state(), o.state(), c)
        assert max(r) <= TOL_ONE_STEP, (p_shock, r)
    s0.close()
    o.step(59), s.step(59)
    da, db = s.diagnostics(), o.diagnostics()
    assert da["step"] == db["step"] == 60 and da["bad_state"] == 0
    assert da["t"] == pytest.approx(db["t"], rel=1e-11)
    assert da["M2r"] == pytest.approx(db["M2r"], rel=1e-11)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= TOL_L1_500, l1
    # the shocked slab sits at the input pressure (the three runs really differ)
    assert o.read_field("p")[:, :60].mean() == pytest.approx(p_shock, rel=2e-2)
    _one_step_from(O, B, cfg, o, "C4 crop at %.0f GPa after 60 steps" % (p_shock / 1e9), variants=(0, 1))
    s.close()


@pytest.mark.slow
def test_c4_full_size_500_steps(O, B):
    """BASELINE config 4 at its own size, 8192 x 1024 with ~480 random cavities (phi = 3 %, d = 24 cells, seed 12345), 8 GPa:
    cavity list bit-identical, one step <= 1e-11, 500 free-running steps L1 <= 1e-7 (north_star; SURVEY 8(d) "Parity workload").
    4.2e9 oracle cell-updates: about 280 s on the 16 host threads of the GPU box, the longest test of the suite."""
    cfg = inputs.config("C4")
    o, s = _start(O, B, cfg)
    s_gen = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    s_gen.init(cfg["init"])
    assert np.array_equal(s_gen.cavities(), o.cavities()) and 400 < len(o.cavities()) < 600
    s_gen.close()
    o.step(1), s.step(1)
    r = rel_diff(s.state(), o.state(), o.read_field("c"))
    assert max(r) <= TOL_ONE_STEP, r
    o.step(499), s.step(499)
    da, db = s.diagnostics(), o.diagnostics()
    assert da["step"] == db["step"] == 500 and da["bad_state"] == 0
    assert da["t"] == pytest.approx(db["t"], rel=1e-10)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= TOL_L1_500, l1
    # integrals of two states that differ by L1 <= 1e-7 per field: 1e-9 (measured 1.2e-11 for M2r, the others closer)
    for k in ("M2r", "mass1", "mass2", "momx", "energy"):
        assert da[k] == pytest.approx(db[k], rel=1e-9), k
    assert o.fallback_count() == 0 and s.redo_count() == 0
    print("C4 full, 500 steps: L1 %s" % (["%.1e" % v for v in l1],))
    s.close()


# ------------------------------------------------------------------------------------------------ C5
@pytest.mark.slow
def test_c5_crop_4096x1024_500_steps(O, B):
    """BASELINE config 5's generator parameters (d in U[16, 40], gap 4, phi = 5 %, seed 12345) on the 4096 x 1024 crop
    SURVEY 8(d) names: cavity list bit-identical, one step, 500 steps"""
    cfg = inputs.config("C5", nx=4096, ny=1024)
    o, s = _start(O, B, cfg)
    s_gen = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    s_gen.init(cfg["init"])
    assert np.array_equal(s_gen.cavities(), o.cavities()) and len(o.cavities()) > 200
    s_gen.close()
    o.step(1), s.step(1)
    r = rel_diff(s.state(), o.state(), o.read_field("c"))
    assert max(r) <= TOL_ONE_STEP, r
    o.step(499), s.step(499)
    da, db = s.diagnostics(), o.diagnostics()
    assert da["step"] == db["step"] == 500 and da["bad_state"] == 0
    assert da["t"] == pytest.approx(db["t"], rel=1e-10)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= TOL_L1_500, l1
    assert o.fallback_count() == 0
    print("C5 crop 4096 x 1024, 500 steps: L1 %s" % (["%.1e" % v for v in l1],))
