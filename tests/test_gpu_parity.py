"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, same seeded inputs.

Tolerances are BASELINE.json north_star's, all fp64: max relative difference in every conserved variable
<= 1e-11 after one step (metric R18, tests/parity_util.py), L1-relative <= 1e-7 after 500 steps, global
reaction-rate curve and overtake time within 0.5 %.  Integer work (cavity list) is bit-exact.
Oracle inputs never come from the CUDA path: states are produced by the oracle and handed to the GPU.
"""
import numpy as np
import pytest

from paper_1905_05727_b200 import inputs
from parity_util import TOL_L1_500, TOL_ONE_STEP, TOL_RATE, l1_rel, rel_diff

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1905_05727_b200 import binding, build
    build.build()                   # no-op when libnmsdt.so is up to date (nvcc cross-compiles sm_100a in ~20 s otherwise)
    binding.load_library()
    return binding


def _pair(O, B, cfg, threads=8, variant=None):
    o = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=threads)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant)
    return o, s


def _sync_state(o, s):
    """hand the oracle's state to the GPU"""
    s.init_fields(o.state())


def _assert_one_step(o, s, tol=TOL_ONE_STEP, what=""):
    qa, qb = s.state(), o.state()
    r = rel_diff(qa, qb, o.read_field("c"))
    assert max(r) <= tol, "%s rel diff per variable %s" % (what, r)
    return r


VARIANTS = [0, 1]


# ------------------------------------------------------------------------------------------------ init
def test_init_fields_round_trip_is_exact(O, B):
    cfg = inputs.config("C1")
    o, s = _pair(O, B, cfg)
    o.init(cfg["init"])
    _sync_state(o, s)
    for a, b in zip(s.state(), o.state()):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("name,kw", [("C1", {}), ("C3", dict(nx=1024, ny=256)), ("C4", dict(nx=2048, ny=512)),
                                     ("C5", dict(nx=2048, ny=512))])
def test_sim_init_matches_oracle_init(O, B, name, kw):
    cfg = inputs.config(name, **kw)
    o, s = _pair(O, B, cfg)
    o.init(cfg["init"])
    s.init(cfg["init"])
    ca, cb = s.cavities(), o.cavities()
    assert ca.shape == cb.shape and np.array_equal(ca, cb)          # integer work: bit-exact
    qa, qb = s.state(), o.state()
    for k in range(7):
        # q1, q6 carry z2 = 1 - z1: where z1 -> 1 - 1e-6 one ulp of tanh is 1e-10 of z2
        np.testing.assert_allclose(qa[k], qb[k], rtol=1e-12, atol=1e-12 if k in (1, 6) else 0)
    da, db = s.diagnostics(), o.diagnostics()
    assert da["M2tot0"] == pytest.approx(db["M2tot0"], rel=1e-12)
    assert s.cfl_dt() == pytest.approx(o.cfl_dt(), rel=1e-13)


def test_generator_matches_oracle_at_full_c4_and_c5_sizes(O, B):
    for name in ("C4", "C5"):
        cfg = inputs.config(name)
        ini, g = cfg["init"], cfg["grid"]
        ref = O.gen_cavities(ini["seed"], ini["phi"], ini["dmin"], ini["dmax"], ini["min_gap"], ini["x_lo"], ini["x_hi"],
                             g["ny"], 1)
        # drive only the generator: a grid with the real ny but few columns would change x_hi, so use a thin
        # dummy grid and the explicit generator parameters through sim_init on a narrow strip is not possible;
        # C4 fits easily, C5's generator is checked on the full grid in test_full_size_sampled_parity.
        if name == "C4":
            s = B.Sim(g, cfg["eos"], cfg["kin"])
            s.init(ini)
            assert np.array_equal(s.cavities(), ref)
            assert 400 < len(ref) < 600
            s.close()
        else:
            assert 8000 < len(ref) < 13000


def test_out_of_range_volume_fraction_is_clamped_on_entry_by_both_sides(O, B):
    """R27: sim_init_fields and orc_init_fields both store q5 clamped to [z_min, 1 - z_min]; a buffer with q5 outside (0, 1,
    beyond) gives the same stored state and the same first step on both sides, in both variants."""
    cfg, o0 = _developed_c1(O, reactive=1, steps=200)
    q = [a.copy() for a in o0.state()]
    rng = np.random.default_rng(5)
    zmin = cfg["eos"]["z_min"]
    # out-of-range values only where the clamp returns (nearly) the value the developed state holds, so that the clamped
    # state is a state of the scheme: pure liquid (q5 = z_min) -> 0, negative, 1e-9; cavity interior (q5 >= 1 - 2 z_min) -> 1, 1.2
    lo, hi = np.flatnonzero(q[5].ravel() == zmin), np.flatnonzero(q[5].ravel() >= 1.0 - 2.0 * zmin)
    assert lo.size > 1000
    pick = rng.choice(lo, 300, replace=False)
    q[5].ravel()[pick] = rng.choice([0.0, -0.1, 1e-9], 300)
    if hi.size:
        q[5].ravel()[hi] = rng.choice([1.0, 1.2, 1.0 - 1e-9], hi.size)
    for variant in VARIANTS:
        o, s = _pair(O, B, cfg, variant=variant)
        o.init_fields(q)
        s.init_fields(q)
        for a, b in zip(s.state(), o.state()):
            assert np.array_equal(a, b)
        assert s.state()[5].min() == zmin and s.state()[5].max() <= 1.0 - zmin
        assert np.array_equal(s.state()[5].ravel()[pick], np.full(300, zmin))
        dt = o.cfl_dt()
        assert s.cfl_dt() == pytest.approx(dt, rel=1e-13)
        o.step_dt(1, 0.25 * dt)
        s.step_dt(1, 0.25 * dt)
        _assert_one_step(o, s, what="clamped entry state, variant %d" % variant)
        s.close()


# ------------------------------------------------------------------------------------------------ pieces
def _developed_c1(O, reactive, steps=120, threads=8):
    cfg = inputs.config("C1", reactive=reactive)
    o = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=threads)
    o.init(cfg["init"])
    o.step(steps)
    return cfg, o


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("d", [0, 1])
def test_single_sweep_parity(O, B, d, variant):
    cfg, o = _developed_c1(O, reactive=0, steps=400)       # shock inside the cavity: strong 2D structure
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant)
    _sync_state(o, s)
    dt = o.cfl_dt()
    o.sweep(d, dt)
    s.sweep(d, dt)
    _assert_one_step(o, s, what="sweep dir %d" % d)
    assert o.fallback_count() == 0


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("bc", [0, 1, 2, 3])
def test_halo_rules_through_sweeps(O, B, bc, variant):
    # a small box whose activity touches every boundary; ragged sizes (not multiples of any tile)
    nx, ny = 83, 37
    bcx = (bc, bc if bc != 3 else 0)
    bcy = (bc if bc != 3 else 1,) * 2
    grid = dict(nx=nx, ny=ny, dx=4e-6, dy=4e-6, bc_xlo=bcx[0], bc_xhi=bcx[1], bc_ylo=bcy[0], bc_yhi=bcy[1], cfl=0.4, limiter=0)
    kin = dict(inputs.KIN, reactive=0)
    ini = dict(inputs._INIT0, p_shock=9e9, shock_cells=6, cavities=[(2.0, 3.0, 7.0), (80.0, 35.0, 6.0), (40.0, 0.0, 5.0)])
    o = O.Oracle(grid, inputs.EOS, kin)
    o.init(ini)
    s = B.Sim(grid, inputs.EOS, kin, variant=variant)
    _sync_state(o, s)
    for it in range(6):                 # no re-sync: both sides keep their own state and step parity
        dt = o.cfl_dt()
        assert s.cfl_dt() == pytest.approx(dt, rel=1e-12)
        o.step_dt(1, dt)
        s.step_dt(1, dt)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="bc %d step %d" % (bc, it))


@pytest.mark.parametrize("variant", VARIANTS)
def test_source_step_parity(O, B, variant):
    cfg, o = _developed_c1(O, reactive=1, steps=400)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant)
    _sync_state(o, s)
    for tau in (1e-10, 5e-9):           # 5e-9: forces several RK4 sub-steps in the hot cells
        o.source(tau)
        s.source(tau)
        r = _assert_one_step(o, s, what="source tau=%g" % tau)
        _sync_state(o, s)
    assert o.read_field("lambda")[:, 40:].min() < 0.999     # something burned outside the inert slab


@pytest.mark.parametrize("variant", VARIANTS)
def test_diagnostics_and_cfl_parity(O, B, variant):
    cfg, o = _developed_c1(O, reactive=1, steps=300)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant)
    o2 = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"])
    o2.init(cfg["init"])
    s.init(cfg["init"])
    m0 = s.diagnostics()["M2tot0"]
    _sync_state(o, s)
    assert s.cfl_dt() == pytest.approx(o.cfl_dt(), rel=1e-13)
    da, db = s.diagnostics(), o.diagnostics()
    for k in ("M2r", "mass1", "mass2", "momx", "energy", "rate_inst", "smax"):
        assert da[k] == pytest.approx(db[k], rel=1e-12), k
    assert abs(da["momy"] - db["momy"]) <= 1e-12 * abs(db["momx"])
    assert da["bad_state"] == 0
    # deterministic reduction: same bits twice
    assert s.diagnostics() == da


def test_derived_fields_parity(O, B):
    cfg, o = _developed_c1(O, reactive=1, steps=200)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"])
    _sync_state(o, s)
    for name, tol in (("p", 1e-9), ("T2", 1e-9), ("rho", 1e-14), ("u", 1e-13), ("v", 1e-13), ("lambda", 1e-13),
                      ("progress", 1e-13), ("rho2", 1e-13), ("c", 1e-10), ("rho1", 1e-13), ("T1", 1e-9)):
        a, b = s.read_field(name), o.read_field(name)
        scale = np.maximum(np.abs(b), np.max(np.abs(b)) * 1e-6 + 1e-300)
        assert np.max(np.abs(a - b) / scale) < tol, name


def test_bad_state_is_reported(O, B):
    cfg = inputs.config("C1")
    o, s = _pair(O, B, cfg)
    o.init(cfg["init"])
    q = o.state()
    q[4][5, 7] = np.nan
    s.init_fields(q)
    with pytest.raises(B.NmsdtError) as e:
        s.cfl_dt()
    assert e.value.code == B.SIM_ERR_BAD
    assert s.diagnostics(allow_bad=True)["bad_state"] == 1


# ------------------------------------------------------------------------------------------------ whole steps
ONE_STEP_CASES = [
    ("C1", dict(reactive=0), 0), ("C1", dict(reactive=1), 0), ("C1", dict(reactive=1), 400),
    ("C2", dict(nx=1024, ny=32, p_shock=11e9), 0), ("C2", dict(nx=1024, ny=8, p_shock=11e9), 1500),
    ("C3", dict(nx=768, ny=192), 0), ("C4", dict(nx=1536, ny=384), 0), ("C5", dict(nx=1536, ny=384), 0),
]


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("name,kw,pre", ONE_STEP_CASES)
def test_one_step_parity(O, B, name, kw, pre, variant):
    cfg = inputs.config(name, **kw)
    o, s = _pair(O, B, cfg, variant=variant)
    o.init(cfg["init"])
    t_pre = 0.0
    if pre:
        o.step(pre)
        t_pre = o.diagnostics()["t"]
        o2 = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=8)     # restart the step counter at 0 on both sides
        o2.init_fields(o.state())
        o, t_pre = o2, 0.0
    _sync_state(o, s)
    for it in range(2):                 # an even (X-Y) and an odd (Y-X) step; no re-sync in between
        dt = o.cfl_dt()
        o.step(1)
        s.step(1)                       # the GPU takes its own device-side CFL dt
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="%s %s pre=%d step %d" % (name, kw, pre, it))
        da, db = s.diagnostics(), o.diagnostics()
        assert da["dt_last"] == pytest.approx(dt, rel=1e-12) and da["step"] == it + 1
        assert da["t"] == pytest.approx(db["t"] - (0.0 if not pre else t_pre), rel=1e-12)
    assert o.fallback_count() == 0


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("reactive", [0, 1])
def test_one_step_parity_mc_limiter(O, B, reactive, variant):
    """the switchable monotonised-central limiter (R5), reactive and inert (the fused path has kernels of its own for
    each limiter and for inert runs)"""
    cfg = inputs.config("C1", reactive=reactive)
    o0 = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=8)
    o0.init(cfg["init"])
    o0.step(400)
    cfg["grid"]["limiter"] = inputs.LIM_MC
    o, s = _pair(O, B, cfg, variant=variant)
    o.init_fields(o0.state())
    _sync_state(o, s)
    for it in range(2):
        o.step(1)
        s.step(1)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="MC limiter step %d" % it)
    o_mm = O.Oracle(dict(cfg["grid"], limiter=inputs.LIM_MINMOD), cfg["eos"], cfg["kin"], threads=8)
    o_mm.init_fields(o0.state())
    o_mm.step(2)
    assert max(rel_diff(o_mm.state(), o.state(), o.read_field("c"))) > 1e-6      # the limiter really differs


@pytest.mark.parametrize("variant", VARIANTS)
def test_rare_paths_substepped_source_inside_full_steps(O, B, variant):
    """R13 inside sim_step: with theta_0 lowered to 2e-5 every shocked cell needs several RK4 sub-steps, so the fused
    kernels take their redo path (a warp whose segment holds such a cell repeats it with the exact rule)."""
    cfg = inputs.config("C1", reactive=1)
    o0 = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=8)
    o0.init(cfg["init"])
    o0.step(400)
    cfg["kin"]["substep_theta"] = 2e-5
    o, s = _pair(O, B, cfg, variant=variant)
    o.init_fields(o0.state())
    _sync_state(o, s)
    e = O.make_eos(cfg["eos"]); k = O.make_kin(cfg["kin"])
    q = np.array([f[64, 20] for f in o.state()])                 # a cell of the shocked slab's wake
    assert O.source_cell(e, k, q, 0.5 * o.cfl_dt())[1] > 1       # the rule really asks for sub-steps there
    for it in range(2):
        o.step(1)
        s.step(1)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="substepped step %d" % it)


@pytest.mark.parametrize("patch", [(30, 150, 2.0, 1.0e5), (90, 200, 3.4e5, 1.0e20)])
def test_rare_paths_density_outside_the_power_tables(O, B, patch):
    """The fused kernels take x^C, x^D of Eq. 3-4 (x = rho2/rho02) from binade tables that cover 2^-8 <= x < 2^8; a cell or
    a reconstructed face outside makes the warp redo its segment with the library powers.  A patch of very dilute
    (x = 1.8e-3) or very dense (x = 300; its pressure is of the size of p_ref(x) ~ 1e20 Pa so that Eq. 2 does not cancel)
    liquid inside single sweeps of both directions and inside full steps."""
    cfg = inputs.config("C1", reactive=1)
    o, s = _pair(O, B, cfg, variant=1)
    o.init(cfg["init"])
    o.step(150)
    q = o.state()
    e = O.make_eos(cfg["eos"])
    for (j0, i0, rho2, p) in (patch,):
        for j in range(j0, j0 + 3):
            for i in range(i0, i0 + 3):
                c = O.prim_to_cons(e, np.array([1.2, rho2, 0.0, 0.0, p, 0.3, 1.0]))
                for k in range(7):
                    q[k][j, i] = c[k]
    o.init_fields(q)
    _sync_state(o, s)
    dt = 0.2 * o.cfl_dt()
    for d in (0, 1):
        o.sweep(d, dt), s.sweep(d, dt)
        _assert_one_step(o, s, what="sweep %d with densities outside the tables" % d)
    o.init_fields(q)
    _sync_state(o, s)
    for it in range(2):
        o.step_dt(1, dt), s.step_dt(1, dt)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="step %d with densities outside the tables" % it)
    assert s.diagnostics()["bad_state"] == 0


@pytest.mark.parametrize("variant", VARIANTS)
def test_rare_paths_reactant_mass_outside_its_bounds(O, B, variant):
    """O3 clamps lambda = q6/q1 to [0, 1] and O5 moves q1 Q (lambda_0 - lambda_1) with that clamped lambda_0.  Cells planted
    with q6 > q1 and with q6 < 0 (in the hot wake, where the source step is active, and in cold liquid) must come out of the
    leading source step (fused: applied on load, pass 1) as the oracle's do; after the step every lambda is inside again."""
    cfg, o = _developed_c1(O, reactive=1, steps=400)
    q = o.state()
    rng = np.random.default_rng(5)
    for (j0, i0) in ((20, 10), (64, 20), (100, 60), (64, 200), (5, 250)):
        for j in range(j0, j0 + 4):
            for i in range(i0, i0 + 4):
                f = rng.choice([1.0 + 1e-3, 1.2, -1e-3, -0.3, 1.0 + 1e-15])
                q[6][j, i] = f * q[1][j, i]
    o2, s = _pair(O, B, cfg, variant=variant)
    o2.init_fields(q)
    _sync_state(o2, s)
    for it in range(2):
        o2.step(1), s.step(1)
        _assert_one_step(o2, s, tol=(it + 1) * TOL_ONE_STEP, what="planted q6, step %d" % it)
    assert s.diagnostics()["bad_state"] == 0
    lam = o2.read_field("lambda")
    assert lam.min() >= 0.0 and lam.max() <= 1.0


@pytest.mark.parametrize("nx,ny", [(255, 64), (257, 31), (4093, 8), (2051, 5)])
def test_odd_nx_takes_the_fast_path(O, B, nx, ny):
    """Rows with an odd number of cells end in a pair whose second cell is row padding: the x-sweep must neither store nor
    act on what it computes from it (no redo of the row's last segment), and still match the oracle."""
    cfg = inputs.config("C4", nx=nx, ny=ny, p_shock=9e9)
    o, s = _pair(O, B, cfg, variant=1)
    o.init(cfg["init"])
    o.step(60)
    _sync_state(o, s)
    for it in range(4):
        o.step(1), s.step(1)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="odd nx %d step %d" % (nx, it))
    assert s.redo_count() == 0
    # ... while a run that needs the exact rules does count (theta_0 lowered: every shocked cell sub-steps)
    cfg["kin"]["substep_theta"] = 2e-5
    s2 = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=1)
    s2.init_fields(o.state())
    s2.step(1)
    assert s2.redo_count() > 0


def test_generator_reports_the_air_fraction_it_placed(O, B):
    """R16: the seeded generator stops at the target air fraction; a target at the jamming limit of the minimum gap is an
    error, not a silently thinner field (the paper's densest case, phi = 8 % with centre spacing 2.5 d_c, is
    reachable and must be reached)"""
    cfg = inputs.paper_case("random", dx_um=8.0, phi=0.08)
    g, ini = cfg["grid"], cfg["init"]
    s = B.Sim(g, cfg["eos"], cfg["kin"])
    s.init(ini)
    want, got = s.cavity_stats()
    cav = s.cavities()
    area = (ini["x_hi"] - ini["x_lo"]) * g["ny"]
    assert want == 0.08 and got >= 0.08 and got == pytest.approx(np.pi * np.sum(cav[:, 2] ** 2) / area, rel=1e-12)
    assert got - 0.08 < np.pi * cav[0, 2] ** 2 / area                  # stops with the cavity that reaches the target
    ref = O.gen_cavities(ini["seed"], ini["phi"], ini["dmin"], ini["dmax"], ini["min_gap"], ini["x_lo"], ini["x_hi"], g["ny"], 1)
    assert np.array_equal(cav, ref)
    # Eq. 8: N = 4 phi L W / (pi d_c^2)
    assert len(cav) == int(np.ceil(4 * 0.08 * area / (np.pi * ini["dmin"] ** 2)))
    ini_bad = dict(ini, phi=0.12)                                       # exclusion disks would cover 0.75 of the plane: beyond jamming
    with pytest.raises(B.NmsdtError) as e:
        s.init(ini_bad)
    assert e.value.code == B.SIM_ERR_ARG and "air fraction" in str(e.value)
    want, got = s.cavity_stats()
    assert want == 0.12 and 0.08 < got < 0.10
    with pytest.raises(B.NmsdtError):
        s.step(1)                                                       # the failed init left no usable state
    s.init(ini)
    s.step(2)
    assert s.diagnostics()["bad_state"] == 0


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("d", [0, 1])
def test_rare_paths_first_order_fallback(O, B, d, variant):
    """R17: the scheme never needs the fallback at CFL 0.4 (nor at 10x that step); a sweep with 40x (x) / 160x (y) the
    CFL step on a developed cavity collapse predicts non-positive face densities in some cells, and both sides must
    fall back to first order in exactly those cells.  The input state is valid, so every output is finite."""
    cfg, o = _developed_c1(O, reactive=0, steps=600)
    s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=variant)
    _sync_state(o, s)
    mult = 40.0 if d == 0 else 160.0
    dt = mult * o.cfl_dt()
    n0 = o.fallback_count()
    c_before = o.read_field("c")
    o.sweep(d, dt)
    s.sweep(d, dt)
    assert o.fallback_count() > n0, "the case must trigger the fallback"
    qa, qb = s.state(), o.state()
    assert all(np.isfinite(a).all() for a in qa) and all(np.isfinite(b).all() for b in qb)
    r = rel_diff(qa, qb, c_before)                                # sound speed of the (valid) input state as the momentum scale
    # the update is q - (dt/dx) dF: the rounding differences of the fluxes are amplified by the step multiplier (a
    # cell that fell back on one side only would differ by ~1e-2)
    assert max(r) <= mult * TOL_ONE_STEP, r


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("ratio", [0.7, 1.6])
def test_non_square_cells(O, B, ratio, variant):
    """dy = ratio * dx: the y-sweep's dt/dy, the CFL step's min(dx, dy) (R11) and the diagnostics' dx dy, on a developed
    cavity collapse (the oracle side is pinned on such grids by tests/test_oracle_cfl.py)"""
    cfg, o0 = _developed_c1(O, reactive=1, steps=400)
    g = dict(cfg["grid"], dy=ratio * cfg["grid"]["dx"])
    o = O.Oracle(g, cfg["eos"], cfg["kin"], threads=8)
    o.init_fields(o0.state())
    s = B.Sim(g, cfg["eos"], cfg["kin"], variant=variant)
    _sync_state(o, s)
    dt = o.cfl_dt()
    assert s.cfl_dt() == pytest.approx(dt, rel=1e-13)
    assert dt == pytest.approx(0.4 * min(g["dx"], g["dy"]) / o.diagnostics()["smax"], rel=1e-13)
    for d in (0, 1):
        o.sweep(d, dt), s.sweep(d, dt)
        _assert_one_step(o, s, what="sweep %d, dy = %g dx" % (d, ratio))
        o.init_fields(o0.state())
        _sync_state(o, s)
    for it in range(2):
        o.step(1), s.step(1)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="step %d, dy = %g dx" % (it, ratio))
    da, db = s.diagnostics(), o.diagnostics()
    for k in ("t", "dt_last", "M2r", "mass1", "mass2", "momx", "energy", "rate_inst", "smax"):
        assert da[k] == pytest.approx(db[k], rel=1e-12), k
    # the cell shape matters: the same two steps on square cells give another state
    o_sq = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"], threads=8)
    o_sq.init_fields(o0.state())
    o_sq.step(2)
    assert max(rel_diff(o_sq.state(), o.state(), o.read_field("c"))) > 1e-4


@pytest.mark.parametrize("variant", VARIANTS)
def test_500_steps_l1_parity_c1(O, B, variant):
    cfg = inputs.config("C1", reactive=1)
    o, s = _pair(O, B, cfg, variant=variant)
    o.init(cfg["init"])
    s.init(cfg["init"])
    o.step(500)
    s.step(500)
    da, db = s.diagnostics(), o.diagnostics()
    assert da["step"] == db["step"] == 500
    assert da["t"] == pytest.approx(db["t"], rel=1e-9)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= TOL_L1_500, l1
    assert o.fallback_count() == 0


@pytest.mark.parametrize("variant", VARIANTS)
def test_500_steps_l1_parity_random_cavities_crop(O, B, variant):
    cfg = inputs.config("C4", nx=768, ny=192)
    o, s = _pair(O, B, cfg, variant=variant)
    o.init(cfg["init"])
    s.init(cfg["init"])
    assert len(o.cavities()) >= 5
    o.step(500)
    s.step(500)
    l1 = l1_rel(s.state(), o.state())
    assert max(l1) <= TOL_L1_500, l1


def test_reaction_rate_curve_and_overtake_time(O, B):
    # neat NM strip (C2 shape, cropped so the oracle finishes in seconds), 11 GPa: ignition within ~0.3 us
    cfg = inputs.config("C2", nx=1024, ny=4, p_shock=11e9)
    o, s = _pair(O, B, cfg, variant=1)
    o.init(cfg["init"])
    s.init(cfg["init"])
    ta, Ma, tb, Mb = [0.0], [s.diagnostics()["M2r"]], [0.0], [o.diagnostics()["M2r"]]
    for _ in range(220):                # sample every 10 steps (R14)
        o.step(10)
        s.step(10)
        da, db = s.diagnostics(), o.diagnostics()
        ta.append(da["t"]); Ma.append(da["M2r"]); tb.append(db["t"]); Mb.append(db["M2r"])
    ta, Ma, tb, Mb = map(np.array, (ta, Ma, tb, Mb))
    ra = np.abs(np.diff(Ma)) / np.diff(ta) / da["M2tot0"]
    rb = np.abs(np.diff(Mb)) / np.diff(tb) / db["M2tot0"]
    k = int(np.argmax(rb))
    assert 20 < k < len(rb) - 5, "rate peak must lie inside the run (k=%d)" % k
    sig = rb > 0.01 * rb[k]
    assert np.max(np.abs(ra[sig] / rb[sig] - 1.0)) < TOL_RATE
    t_a, t_b = 0.5 * (ta[1:] + ta[:-1])[int(np.argmax(ra))], 0.5 * (tb[1:] + tb[:-1])[k]
    assert t_a == pytest.approx(t_b, rel=TOL_RATE)


# ------------------------------------------------------------------------------------------------ full size
@pytest.mark.parametrize("name", ["C3", "C4", "C5"])
def test_full_size_sampled_parity(O, B, name):
    """BASELINE.json's full sizes in the launch configuration bench.py times: the GPU advances the whole grid,
    the oracle recomputes sampled windows (window + 8-cell margin = 2 steps x 2 sweeps x radius 2)."""
    cfg = inputs.config(name)
    g = cfg["grid"]
    s = B.Sim(g, cfg["eos"], cfg["kin"], variant=1)
    s.init(cfg["init"])
    cav = s.cavities()
    if name != "C3":
        ini = cfg["init"]
        ref = O.gen_cavities(ini["seed"], ini["phi"], ini["dmin"], ini["dmax"], ini["min_gap"], ini["x_lo"], ini["x_hi"], g["ny"], 1)
        assert np.array_equal(cav, ref)
    d0 = s.diagnostics()
    dt = 0.9 * s.cfl_dt()
    nx, ny = g["nx"], g["ny"]
    W, M = 48, 8
    rng = np.random.default_rng(2024)
    wins = [(96, 0), (nx - W - 2 * M, ny - W - 2 * M)]                 # shock front; far corner
    for c in cav[rng.choice(len(cav), size=3, replace=False)]:          # around cavities
        wins.append((int(np.clip(c[0] - W // 2 - M, 0, nx - W - 2 * M)), int(np.clip(c[1] - W // 2 - M, 0, ny - W - 2 * M))))
    before = s.state()
    s.step_dt(2, dt)
    after = s.state()
    d1 = s.diagnostics()
    assert d1["step"] == 2 and d1["t"] == pytest.approx(2 * dt, rel=1e-14)
    for (x0, y0) in wins:
        sl = (slice(y0, y0 + W + 2 * M), slice(x0, x0 + W + 2 * M))
        wg = dict(g, nx=W + 2 * M, ny=W + 2 * M, bc_xlo=0, bc_xhi=0, bc_ylo=0, bc_yhi=0)
        o = O.Oracle(wg, cfg["eos"], cfg["kin"])
        o.init_fields([a[sl] for a in before])
        o.step_dt(2, dt)
        qa = [a[sl][M:-M, M:-M] for a in after]
        qb = [b[M:-M, M:-M] for b in o.state()]
        r = rel_diff(qa, qb, o.read_field("c")[M:-M, M:-M])
        assert max(r) <= 2 * TOL_ONE_STEP, "%s window %s: %s" % (name, (x0, y0), r)
    # global invariants that hold at any size: phase masses change only through the x boundaries (inflow)
    assert d1["mass2"] > d0["mass2"] and d1["bad_state"] == 0
    assert abs(d1["momy"]) < 1e-9 * abs(d1["momx"]) or name != "C3"


# ------------------------------------------------------------------------------------------------ launch geometry
@pytest.mark.parametrize("name,kw", [("C1", {}), ("C2", {}), ("C3", {}), ("C4", {}), ("C5", {}), ("C4", dict(nx=83, ny=37))])
def test_sweep_geometry_covers_the_grid(B, name, kw):
    """sim_sweep_geometry: every cell belongs to exactly one segment; grids that fill the GPU get long segments (little ramp-up
    redundancy), grids that cannot are cut short (latency of the march is what counts there)"""
    cfg = inputs.config(name, **kw)
    g = cfg["grid"]
    s = B.Sim(g, cfg["eos"], cfg["kin"])
    for d, (n, lines) in enumerate(((g["nx"], (g["ny"] + 3) // 4), (g["ny"], (g["nx"] + 255) // 256))):
        seg, ramp, nb = s.sweep_geometry(d)
        assert seg >= 1 and ramp == 4 and nb == lines * ((n + seg - 1) // seg)
        if d == 0:
            assert (seg + ramp) % 64 == 0 and seg % 2 == 0                  # whole 64-cell chunks, even starts (pair loads)
        if name == "C5" and not kw:
            assert (seg + ramp) / seg < 1.02 and nb > 8 * 148
        if name in ("C1",) and not kw:
            assert nb <= 148 * 4 and seg <= (60 if d == 0 else 4)
    s.close()


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("nx,ny,bcx,bcy", [(8, 8, 1, 1), (2, 2, 1, 1), (2, 3, 0, 2), (5, 1, 2, 1), (1, 6, 0, 0), (63, 2, 3, 1), (66, 4, 2, 2)])
def test_tiny_grids(O, B, nx, ny, bcx, bcy, variant):
    """grids smaller than one chunk / one segment, down to a single row or column: every cell's stencil reaches a ghost cell, so
    the boundary rules folded into the sweeps (periodic wrap of 1- and 2-cell lines, mirror images, fixed inflow) carry the result"""
    bx = (bcx, bcx if bcx != 3 else 0)
    grid = dict(nx=nx, ny=ny, dx=4e-6, dy=4e-6, bc_xlo=bx[0], bc_xhi=bx[1], bc_ylo=bcy, bc_yhi=bcy, cfl=0.4, limiter=0)
    rng = np.random.default_rng(100 * nx + ny)
    e = O.make_eos(inputs.EOS)
    q = np.empty((7, ny, nx))
    for j in range(ny):
        for i in range(nx):
            W = [1.2 * rng.uniform(1, 30), 1134.0 * rng.uniform(1.0, 1.6), rng.uniform(-800, 800), rng.uniform(-800, 800),
                 10 ** rng.uniform(5, 9.9), rng.choice([1e-6, 0.3, 1 - 1e-6]), rng.uniform(0.2, 1.0)]
            q[:, j, i] = O.prim_to_cons(e, np.array(W))
    o = O.Oracle(grid, inputs.EOS, inputs.KIN)
    o.init_fields(list(q))
    s = B.Sim(grid, inputs.EOS, inputs.KIN, variant=variant)
    s.init_fields(list(q))
    for it in range(4):
        dt = 0.5 * o.cfl_dt()
        o.step_dt(1, dt), s.step_dt(1, dt)
        _assert_one_step(o, s, tol=(it + 1) * TOL_ONE_STEP, what="tiny %dx%d bc %d/%d step %d" % (nx, ny, bcx, bcy, it))
    assert s.diagnostics()["bad_state"] == 0


def test_launch_modes_change_nothing_but_timing(B):
    """sim_set_launch_mode: CUDA-graph replay and programmatic dependent launch reorder when kernels start, never what they
    compute: 11 steps (odd: the graph path replays pairs and enqueues the rest) give bit-identical states in all four modes"""
    cfg = inputs.config("C4", nx=640, ny=160, p_shock=9e9)
    ref = None
    for use_graph in (True, False):
        for use_pdl in (False, True):
            s = B.Sim(cfg["grid"], cfg["eos"], cfg["kin"], variant=1)
            s.set_launch_mode(use_graph=use_graph, use_pdl=use_pdl)
            s.init(cfg["init"])
            s.step(4)
            s.step(7)
            q = s.state()
            d = s.diagnostics()
            assert d["step"] == 11 and d["bad_state"] == 0
            if ref is None:
                ref = (q, d)
            else:
                assert all(np.array_equal(a, b) for a, b in zip(q, ref[0])) and d == ref[1], (use_graph, use_pdl)
            s.close()
