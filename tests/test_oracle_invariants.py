"""Scheme invariants that pin the oracle's sweep / halo / step (BASELINE.json north_star):
uniform state preserved, pressure-velocity-equilibrium interface advected without spurious p,u,
exact conservation in a closed (periodic / reflective) box, reactive energy bookkeeping, symmetry,
HLLC consistency, limiter properties.
"""
import numpy as np
import pytest

from paper_1905_05727_b200 import inputs

KIN_OFF = dict(inputs.KIN, reactive=0)


def _grid(nx, ny, dx=4e-6, bcx=(1, 1), bcy=(1, 1), limiter=0):
    return dict(nx=nx, ny=ny, dx=dx, dy=dx, bc_xlo=bcx[0], bc_xhi=bcx[1], bc_ylo=bcy[0], bc_yhi=bcy[1], cfl=0.4,
                limiter=limiter)


def _fields_from_prims(O, eos, W):
    """W: (7, ny, nx) primitive arrays -> list of 7 conserved arrays via the oracle's own prim_to_cons."""
    e = O.make_eos(eos)
    ny, nx = W.shape[1:]
    q = np.empty_like(W)
    for j in range(ny):
        for i in range(nx):
            q[:, j, i] = O.prim_to_cons(e, W[:, j, i])
    return list(q)


def _blob_state(nx, ny, rng, u0=300.0):
    """smooth NM/air blob with pressure pulse and velocity field (all positive, well inside the EOS range)"""
    y, x = np.meshgrid((np.arange(ny) + 0.5) / ny, (np.arange(nx) + 0.5) / nx, indexing="ij")
    W = np.empty((7, ny, nx))
    r2 = (x - 0.4) ** 2 + (y - 0.55) ** 2
    W[5] = 1e-6 + (1 - 2e-6) * 0.5 * (1 - np.tanh((np.sqrt(r2) - 0.2) / 0.05))
    W[0] = 1.2 * (1 + 0.3 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y))
    W[1] = 1134.0 * (1 + 0.2 * np.cos(2 * np.pi * (x + y)))
    W[2] = u0 * np.sin(2 * np.pi * y) + 50.0
    W[3] = -u0 * np.cos(2 * np.pi * x)
    W[4] = 1e5 + 2.0e9 * np.exp(-((x - 0.7) ** 2 + (y - 0.3) ** 2) / 0.02)
    W[6] = 0.5 + 0.5 * np.sin(2 * np.pi * x) ** 2
    return W


def test_uniform_state_is_preserved_bitwise(O):
    for bc in (0, 1, 2):
        g = _grid(24, 16, bcx=(bc, bc), bcy=(bc, bc))
        o = O.Oracle(g, inputs.EOS, KIN_OFF)
        W = np.empty((7, 16, 24))
        u0 = 0.0 if bc == 2 else 250.0
        for k, v in enumerate([3.3, 1500.0, u0, -u0 * 0.5, 2.5e9, 0.25, 0.7]):
            W[k] = v
        q = _fields_from_prims(O, inputs.EOS, W)
        o.init_fields(q)
        o.step(7)
        for a, b in zip(o.state(), q):
            assert np.array_equal(a, b)


@pytest.mark.parametrize("limiter", [0, 1])
def test_equilibrium_interface_advects_without_pressure_or_velocity_errors(O, limiter):
    # uniform (u, v, p), uniform phase densities, z1 jump smeared over the grid: p and u must stay uniform
    nx, ny = 64, 8
    o = O.Oracle(_grid(nx, ny, limiter=limiter), inputs.EOS, KIN_OFF)
    x = (np.arange(nx) + 0.5) / nx
    W = np.empty((7, ny, nx))
    W[0], W[1], W[2], W[3], W[4], W[6] = 1.2, 1134.0, 800.0, 0.0, 1.0e5, 1.0
    W[5] = (1e-6 + (1 - 2e-6) * 0.5 * (np.tanh((x - 0.3) / 0.03) - np.tanh((x - 0.6) / 0.03)))[None, :]
    o.init_fields(_fields_from_prims(O, inputs.EOS, W))
    z_int0 = o.read_field("q5").sum()
    n_steps = 0
    while o.diagnostics()["t"] * 800.0 < nx * 4e-6:      # once across the periodic box
        o.step(10)
        n_steps += 10
    p, u, v = o.read_field("p"), o.read_field("u"), o.read_field("v")
    # p is recovered from rho e by cancellation against ~6e8: 1e-16 * 6e8 / 1e5 ~ 1e-12 per operation
    assert np.max(np.abs(p / 1.0e5 - 1.0)) < 1e-7
    assert np.max(np.abs(u / 800.0 - 1.0)) < 1e-10
    assert np.max(np.abs(v)) < 1e-7
    assert np.max(np.abs(o.read_field("rho1") / 1.2 - 1)) < 1e-9
    assert np.max(np.abs(o.read_field("rho2") / 1134.0 - 1)) < 1e-9
    # air volume is conserved and the profile came back to where it started (diffused, not displaced)
    z = o.read_field("q5")
    assert z.sum() == pytest.approx(z_int0, rel=1e-9)
    xc0 = np.sum(W[5][0] * x) / np.sum(W[5][0])
    assert np.sum(z[0] * x) / np.sum(z[0]) == pytest.approx(xc0, abs=1.5 / nx)
    assert z.min() >= 1e-6 and z.max() <= 1 - 1e-6


def test_periodic_box_conserves_mass_momentum_energy_inert(O):
    rng = np.random.default_rng(5)
    nx, ny = 48, 40
    o = O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF)
    o.init_fields(_fields_from_prims(O, inputs.EOS, _blob_state(nx, ny, rng)))
    d0 = o.diagnostics()
    o.step(40)
    d1 = o.diagnostics()
    assert d1["bad_state"] == 0
    for k in ("mass1", "mass2", "energy", "M2r"):
        assert d1[k] == pytest.approx(d0[k], rel=2e-13)
    mom_scale = d0["mass2"] * 300.0
    assert abs(d1["momx"] - d0["momx"]) < 2e-13 * mom_scale
    assert abs(d1["momy"] - d0["momy"]) < 2e-13 * mom_scale
    # and something actually happened
    assert np.max(np.abs(o.read_field("p") - 1e5)) > 1e8 and d1["t"] > 0


def test_reflective_box_conserves_mass_and_energy(O):
    rng = np.random.default_rng(6)
    nx, ny = 40, 32
    o = O.Oracle(_grid(nx, ny, bcx=(2, 2), bcy=(2, 2)), inputs.EOS, KIN_OFF)
    o.init_fields(_fields_from_prims(O, inputs.EOS, _blob_state(nx, ny, rng, u0=100.0)))
    d0 = o.diagnostics()
    o.step(40)
    d1 = o.diagnostics()
    for k in ("mass1", "mass2", "energy"):
        assert d1[k] == pytest.approx(d0[k], rel=2e-13)
    assert abs(d1["momx"] - d0["momx"]) > 1e-6 * abs(d0["mass2"] * 100.0)   # walls do exchange momentum


def test_periodic_box_reactive_conserves_total_plus_chemical_energy(O):
    rng = np.random.default_rng(7)
    nx, ny = 32, 24
    W = _blob_state(nx, ny, rng)
    W[4] = 8e9 + 6.0e9 * np.exp(-((np.arange(nx)[None, :] / nx - 0.7) ** 2) / 0.02)   # hot enough to burn
    W[1] = 1900.0
    o = O.Oracle(_grid(nx, ny), inputs.EOS, inputs.KIN)
    o.init_fields(_fields_from_prims(O, inputs.EOS, W))
    d0 = o.diagnostics()
    o.step(60)
    d1 = o.diagnostics()
    Q = inputs.KIN["Q"]
    assert d0["M2r"] - d1["M2r"] > 1e-4 * d0["M2r"]          # it burned
    assert d1["energy"] + Q * d1["M2r"] == pytest.approx(d0["energy"] + Q * d0["M2r"], rel=5e-13)
    for k in ("mass1", "mass2"):
        assert d1[k] == pytest.approx(d0[k], rel=2e-13)
    assert d1["burned_mass"] == pytest.approx(d0["M2r"] - d1["M2r"], rel=1e-9)
    assert d1["rate_inst"] > 0


def test_mirror_symmetry_of_the_x_sweep(O):
    rng = np.random.default_rng(8)
    nx, ny = 40, 6
    W = _blob_state(nx, ny, rng)
    o1 = O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF)
    o2 = O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF)
    q = _fields_from_prims(O, inputs.EOS, W)
    o1.init_fields(q)
    qm = [a[:, ::-1].copy() for a in q]
    qm[2] = -qm[2]
    o2.init_fields(qm)
    dt = o1.cfl_dt()
    o1.sweep(0, dt)
    o2.sweep(0, dt)
    s1, s2 = o1.state(), o2.state()
    for k in range(7):
        b = s2[k][:, ::-1] * (-1.0 if k == 2 else 1.0)
        scale = np.max(np.abs(s1[k])) + 1e-300
        assert np.max(np.abs(s1[k] - b)) / scale < 1e-13


def test_step_order_alternates_xy_yx(O):
    # R7: even step S X Y S, odd step S Y X S
    rng = np.random.default_rng(9)
    nx, ny = 20, 16
    q = _fields_from_prims(O, inputs.EOS, _blob_state(nx, ny, rng))
    a, b = O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF), O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF)
    a.init_fields(q)
    b.init_fields(q)
    dt = 0.5 * a.cfl_dt()
    a.step_dt(2, dt)
    b.sweep(0, dt); b.sweep(1, dt); b.sweep(1, dt); b.sweep(0, dt)
    for u, v in zip(a.state(), b.state()):
        assert np.array_equal(u, v)


def test_hllc_is_consistent_and_upwinds(O, paper_eos):
    rng = np.random.default_rng(10)
    for _ in range(20):
        W = np.array([rng.uniform(1, 8), rng.uniform(1000, 2200), rng.uniform(-2e3, 2e3), rng.uniform(-1e3, 1e3),
                      10 ** rng.uniform(5, 10), rng.choice([1e-6, 0.4, 1 - 1e-6]), rng.uniform(0, 1)])
        q = O.prim_to_cons(paper_eos, W)
        F, uf = O.hllc(paper_eos, W, W)
        u, p = W[2], W[4]
        Fx = np.array([q[0] * u, q[1] * u, q[2] * u + p, q[3] * u, (q[4] + p) * u, q[5] * u, q[6] * u])
        np.testing.assert_allclose(F, Fx, rtol=1e-12, atol=1e-12 * p)
        assert uf == pytest.approx(u, rel=1e-12, abs=1e-9)
    # supersonic to the right: pure left flux; to the left: pure right flux
    WL = np.array([2.0, 1500.0, 9000.0, 10.0, 1e9, 1e-6, 0.5])
    WR = np.array([1.5, 1300.0, 8800.0, -5.0, 5e8, 1e-6, 0.9])
    F, uf = O.hllc(paper_eos, WL, WR)
    q = O.prim_to_cons(paper_eos, WL)
    assert F[1] == q[1] * WL[2] and uf == WL[2]
    WL[2], WR[2] = -8800.0, -9000.0
    F, uf = O.hllc(paper_eos, WL, WR)
    q = O.prim_to_cons(paper_eos, WR)
    assert F[1] == q[1] * WR[2] and uf == WR[2]


def test_hllc_resolves_isolated_contact_exactly(O, paper_eos):
    # stationary and moving material contact with equal p,u: flux = upwind advection, p,u untouched
    WL = np.array([1.2, 1134.0, 500.0, 0.0, 1e5, 1 - 1e-6, 1.0])
    WR = np.array([1.2, 1134.0, 500.0, 0.0, 1e5, 1e-6, 1.0])
    F, uf = O.hllc(paper_eos, WL, WR)
    q = O.prim_to_cons(paper_eos, WL)
    assert uf == pytest.approx(500.0, rel=1e-12)
    np.testing.assert_allclose(F[[0, 1, 5]], q[[0, 1, 5]] * 500.0, rtol=1e-10)
    assert F[2] == pytest.approx(q[2] * 500.0 + 1e5, rel=1e-10)


def test_limiters(O):
    L = O.lib()
    for kind in (0, 1):
        assert L.orc_limiter(kind, 1.0, -2.0) == 0.0 and L.orc_limiter(kind, 0.0, 3.0) == 0.0
        assert L.orc_limiter(kind, -1.0, -3.0) < 0 and L.orc_limiter(kind, 2.0, 2.0) == 2.0
    assert L.orc_limiter(0, 1.0, 3.0) == 1.0 and L.orc_limiter(0, -4.0, -3.0) == -3.0     # minmod
    assert L.orc_limiter(1, 1.0, 3.0) == 2.0 and L.orc_limiter(1, 1.0, 1.5) == 1.25        # MC


def test_halo_fill_rules(O):
    nx, ny = 6, 5
    rng = np.random.default_rng(11)
    q = [rng.uniform(1, 2, (ny, nx)) for _ in range(7)]
    # the halo itself is observable through one sweep of a transmissive vs periodic box:
    # here check the CFL/diagnostics ignore ghosts and that a periodic shift commutes with a sweep.
    W = np.empty((7, ny, nx))
    for k, v in enumerate([1.2, 1134.0, 100.0, 50.0, 1e5, 0.5, 1.0]):
        W[k] = v
    W[4] = 1e5 * (1 + rng.uniform(0, 1, (ny, nx)))
    qq = _fields_from_prims(O, inputs.EOS, W)
    a, b = O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF), O.Oracle(_grid(nx, ny), inputs.EOS, KIN_OFF)
    a.init_fields(qq)
    b.init_fields([np.roll(np.roll(f, 2, axis=1), 3, axis=0) for f in qq])
    dt = a.cfl_dt()
    assert dt == b.cfl_dt()
    a.step_dt(3, dt)
    b.step_dt(3, dt)
    for u, v in zip(a.state(), b.state()):
        assert np.array_equal(np.roll(np.roll(u, 2, axis=1), 3, axis=0), v)
