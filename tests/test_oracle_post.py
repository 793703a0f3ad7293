"""Pins of the oracle's post-processing: y-averaged profiles Eq. 9-11, the
mass-weighted histogram of the volumetric energy-release rate Eq. 14-16, the leading-shock position and
the moving-averaged shock velocity / acceleration of Appendix C (Eq. C1-C2).

What fixes the expected values: hand-computed averages of a two-row state, the y-uniform special case, mass totals,
the exact bin shift under a rescaling of Q, the oracle's separately pinned rate diagnostic (Eq. 13), the paper's
statements that inert / cold material does not enter the statistics, and the exactness of central differences on a
quadratic trajectory."""
import ctypes as C

import numpy as np
import pytest

from paper_1905_05727_b200 import inputs


def _grid(nx, ny, dx=4e-6):
    return dict(nx=nx, ny=ny, dx=dx, dy=dx, bc_xlo=0, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)


def _sim_from_prims(O, W, kin=None, dx=4e-6):
    """W: (7, ny, nx) primitives (rho1, rho2, u, v, p, z1, lambda) -> oracle holding that state"""
    e = O.make_eos(inputs.EOS)
    ny, nx = W.shape[1:]
    q = np.empty_like(W)
    for j in range(ny):
        for i in range(nx):
            q[:, j, i] = O.prim_to_cons(e, W[:, j, i])
    o = O.Oracle(_grid(nx, ny, dx), inputs.EOS, kin or inputs.KIN)
    o.init_fields(list(q))
    return o


A_ROW = np.array([1.2, 1134.0, 10.0, 0.0, 1e5, 1e-6, 1.0])        # ambient NM
B_ROW = np.array([5.0, 1800.0, 30.0, -7.0, 8e9, 0.3, 0.6])        # compressed NM/air mixture


def test_profiles_two_rows_by_hand(O):
    nx = 4
    W = np.empty((7, 2, nx))
    W[:, 0, :] = A_ROW[:, None]
    W[:, 1, :] = B_ROW[:, None]
    o = _sim_from_prims(O, W)
    pb, rb, ub, xs = o.profiles(1.01e5)
    rho_a = 1e-6 * 1.2 + (1 - 1e-6) * 1134.0
    rho_b = 0.3 * 5.0 + 0.7 * 1800.0
    assert pb == pytest.approx(0.5 * (1e5 + 8e9), rel=1e-9)                       # Eq. 9
    assert rb == pytest.approx(0.5 * (rho_a + rho_b), rel=1e-14)                   # Eq. 10
    assert ub == pytest.approx((rho_a * 10.0 + rho_b * 30.0) / (rho_a + rho_b), rel=1e-13)   # Eq. 11: density weighted,
    assert abs(ub[0] - 20.0) > 0.5                                                 # not the plain mean of u
    assert xs == pytest.approx(nx * 4e-6)                                          # every column is above 1.01 p0


def test_profiles_y_uniform_state_and_front_position(O):
    nx, ny = 12, 5
    W = np.empty((7, ny, nx))
    W[:] = A_ROW[:, None, None]
    W[:, :, :7] = np.array([8.0, 1842.3, 1646.9, 0.0, 8e9, 1e-6, 0.0])[:, None, None]   # shocked slab, 7 columns
    o = _sim_from_prims(O, W, dx=5e-6)
    pb, rb, ub, xs = o.profiles(1.01e5)
    assert np.allclose(pb, o.read_field("p")[2], rtol=1e-12)
    assert np.allclose(rb, o.read_field("rho")[0], rtol=1e-14)
    assert np.allclose(ub, o.read_field("u")[3], rtol=1e-13, atol=1e-9)
    assert xs == pytest.approx(7 * 5e-6, rel=1e-14)             # right edge of the last column with pbar >= 1.01 p0
    assert o.profiles(9e9)[3] == 0.0                            # nothing above the threshold
    # a single shocked cell out of ny rows lifts pbar by (p_s - p0)/ny: the front follows the y-average (R25)
    W[:, 2, 9] = np.array([8.0, 1842.3, 0.0, 0.0, 8e9, 1e-6, 0.0])
    o2 = _sim_from_prims(O, W, dx=5e-6)
    assert o2.profiles(1.01e5)[3] == pytest.approx(10 * 5e-6)
    assert o2.profiles(0.5 * 8e9)[3] == pytest.approx(7 * 5e-6)


def _hot(T_target, O, e, rho2=1850.0, z1=1e-6, lam=1.0):
    """primitive state of NM at density rho2 whose Eq. 5 temperature is T_target (p by bisection on orc_T2)"""
    lo, hi = 1e5, 1e11
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if O.lib().orc_T2(C.byref(e), rho2, mid) < T_target:
            lo = mid
        else:
            hi = mid
    return np.array([8.0, rho2, 0.0, 0.0, 0.5 * (lo + hi), z1, lam])


def test_qdot_pdf_mass_total_bin_from_rate_diagnostic_and_shift(O, paper_eos):
    nx, ny, dx = 6, 4, 4e-6
    W = np.empty((7, ny, nx))
    W[:] = _hot(1500.0, O, paper_eos)[:, None, None]
    o = _sim_from_prims(O, W)
    m, c = o.qdot_pdf(2.0, 0.02, 400)
    d = o.diagnostics()
    # all cells are identical: one bin holds everything; its mass is the NM mass of the domain (z2 rho2 per cell)
    assert c.sum() == nx * ny and (c > 0).sum() == 1
    assert m.sum() == pytest.approx(d["mass2"], rel=1e-13)
    b = int(np.argmax(c))
    # the bin follows from the separately pinned rate diagnostic: qdot = Q * rate_inst / area (Eq. 13-14)
    qdot_gw = inputs.KIN["Q"] * d["rate_inst"] / (nx * ny * dx * dx) / 1e9
    assert 1e2 < qdot_gw < 1e10
    assert 2.0 + 0.02 * b <= np.log10(qdot_gw) < 2.0 + 0.02 * (b + 1)              # Eq. 15
    # magnitude check against Eq. 6 / Table III typed out: rho lam C exp(-Ta/T) Q at 1500 K
    assert qdot_gw == pytest.approx((1 - 1e-6) * 1850.0 * 2.6e9 * np.exp(-11350.0 / 1500.0) * 4.46e6 / 1e9, rel=1e-6)
    # rescaling Q by 10^(k dn) moves every cell by exactly k bins (decadic log scale, Eq. 15)
    for k in (1, 7, -3):
        o2 = _sim_from_prims(O, W, kin=dict(inputs.KIN, Q=inputs.KIN["Q"] * 10 ** (0.02 * k) * (1 + 1e-9)))
        c2 = o2.qdot_pdf(2.0, 0.02, 400)[1]
        assert int(np.argmax(c2)) == b + k and c2.sum() == nx * ny
    # a different window / resolution counts the same cells
    m3, c3 = o.qdot_pdf(0.0, 0.5, 24)
    assert c3.sum() == nx * ny and int(np.argmax(c3)) == int(np.floor(np.log10(qdot_gw) / 0.5))
    # out of the window on either side: nothing counted
    assert o.qdot_pdf(np.log10(qdot_gw) + 0.1, 0.02, 400)[1].sum() == 0
    assert o.qdot_pdf(np.log10(qdot_gw) - 8.1, 0.02, 400)[1].sum() == 0


def test_qdot_pdf_is_mass_weighted_and_skips_inert_and_cold_material(O, paper_eos):
    nx, ny = 8, 3
    W = np.empty((7, ny, nx))
    W[:] = A_ROW[:, None, None]                                       # cold ambient NM: far below 1e2 GW/m^3
    hot1 = _hot(1200.0, O, paper_eos, rho2=1700.0)
    hot2 = _hot(2500.0, O, paper_eos, rho2=2100.0, z1=0.25, lam=0.4)
    inert = _hot(3000.0, O, paper_eos, rho2=1900.0, lam=0.0)          # products (lambda = 0)
    W[:, 0, 0:3] = hot1[:, None]
    W[:, 1, 2:4] = hot2[:, None]
    W[:, 2, 5:8] = inert[:, None]
    o = _sim_from_prims(O, W)
    m, c = o.qdot_pdf(2.0, 0.02, 400)
    dA = 4e-6 ** 2
    assert c.sum() == 5 and sorted(c[c > 0]) == [2, 3]
    b1, b2 = int(np.flatnonzero(c == 3)[0]), int(np.flatnonzero(c == 2)[0])
    assert b2 > b1                                                     # hotter material releases energy faster
    assert m[b1] == pytest.approx(3 * (1 - 1e-6) * 1700.0 * dA, rel=1e-12)          # z2 rho2 dx dy per cell
    assert m[b2] == pytest.approx(2 * 0.75 * 2100.0 * dA, rel=1e-12)
    # an inert run (no kinetics) has no statistics at all
    o_inert = _sim_from_prims(O, W, kin=dict(inputs.KIN, reactive=0))
    assert o_inert.qdot_pdf(2.0, 0.02, 400)[1].sum() == 0


def test_shock_kinematics_exact_on_quadratic_trajectory(O):
    rng = np.random.default_rng(3)
    t = np.sort(np.concatenate([[0.0, 6e-6], rng.uniform(0, 6e-6, 4000)]))          # non-uniform sampling
    x0, u0, a0 = 5e-4, 4300.0, 2.5e8
    xs = x0 + u0 * t + 0.5 * a0 * t * t
    dtau = 1.5e-6                                                                   # the paper's window
    us, acc = O.shock_kinematics(t, xs, dtau)
    inside_u = (t - 0.5 * dtau >= 0) & (t + 0.5 * dtau <= 6e-6)
    inside_a = (t - dtau >= 0) & (t + dtau <= 6e-6)
    assert np.all(np.isnan(us[~inside_u])) and np.all(np.isnan(acc[~inside_a]))
    assert inside_a.sum() > 100
    # central differences are exact for a quadratic; what is left is the linear-interpolation error between samples
    assert np.allclose(us[inside_u], u0 + a0 * t[inside_u], rtol=2e-6)
    assert np.allclose(acc[inside_a], a0, rtol=2e-4)
    # straight trajectory: constant velocity, zero acceleration
    us2, acc2 = O.shock_kinematics(t, x0 + u0 * t, dtau)
    assert np.allclose(us2[inside_u], u0, rtol=1e-12) and np.allclose(acc2[inside_a], 0.0, atol=u0 / dtau * 1e-9)
    # uniform sampling with dtau an even multiple of the spacing: no interpolation at all, Eq. C1 written out
    tu = np.arange(0, 41) * 1e-7
    xu = np.sin(3e5 * tu)
    us3, acc3 = O.shock_kinematics(tu, xu, 4e-7)
    assert us3[10] == pytest.approx((xu[12] - xu[8]) / 4e-7, rel=1e-12)
    assert acc3[10] == pytest.approx((xu[14] - 2 * xu[10] + xu[6]) / 4e-7 ** 2, rel=1e-9)
