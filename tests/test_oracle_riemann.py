"""Pins of the oracle's hydrodynamics (MUSCL-Hancock + limiter + HLLC + non-conservative z1 update)
against exact Riemann solutions (BASELINE.json north_star: Sod and water-air).

The Cochran-Chan form contains the ideal gas (A = B = 0, Gamma2 = gamma-1) and the stiffened gas
(C = D = 0, A = 0, B = p_inf, Gamma2 = gamma_w - 1; energy origin shifted by the constant p_inf/rho0),
so the same oracle code runs both textbook problems.  Exact solutions: tests/riemann_exact.py.
"""
import numpy as np
import pytest

import riemann_exact as RX
from paper_1905_05727_b200 import inputs

KIN_OFF = dict(inputs.KIN, reactive=0)


def _run_tube(O, eos, WL, WR, x0, n, t_end, ny=2, limiter=0, cfl=0.4):
    """1D tube along x on [0,1] (ny identical rows); returns x, fields dict."""
    dx = 1.0 / n
    grid = dict(nx=n, ny=ny, dx=dx, dy=dx, bc_xlo=0, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=cfl, limiter=limiter)
    o = O.Oracle(grid, eos, KIN_OFF)
    e = O.make_eos(eos)
    x = (np.arange(n) + 0.5) * dx
    q = np.empty((7, ny, n))
    qL, qR = O.prim_to_cons(e, WL), O.prim_to_cons(e, WR)
    for k in range(7):
        q[k] = np.where(x < x0, qL[k], qR[k])[None, :]
    o.init_fields(list(q))
    while True:
        dt = o.cfl_dt()
        t = o.diagnostics()["t"]
        if t + dt >= t_end:
            o.step_dt(1, t_end - t)
            break
        o.step_dt(1, dt)
    out = {k: o.read_field(k) for k in ("rho", "u", "v", "p", "q5", "q0", "q1")}
    assert o.fallback_count() == 0
    return x, out, o


def _l1(a, b):
    return np.mean(np.abs(a - b)) / np.mean(np.abs(b))


def test_sod_shock_tube_converges_to_exact_solution(O):
    # both phases the same ideal gas gamma = 1.4; z1 = 0.5 uniform
    eos = dict(inputs.EOS, A=0.0, B=0.0, C=2.0, D=3.0, Gamma2=0.4, rho02=1.0, z_min=1e-6)
    WL = [1.0, 1.0, 0.0, 0.0, 1.0, 0.5, 1.0]
    WR = [0.125, 0.125, 0.0, 0.0, 0.1, 0.5, 1.0]
    errs = []
    for n in (100, 200, 400):
        x, f, _ = _run_tube(O, eos, WL, WR, 0.5, n, 0.2)
        rho, u, p, _ = RX.sample((1.0, 0.0, 1.0, 1.4, 0.0), (0.125, 0.0, 0.1, 1.4, 0.0), (x - 0.5) / 0.2)
        errs.append((_l1(f["rho"][0], rho), np.mean(np.abs(f["u"][0] - u)), _l1(f["p"][0], p)))
        # rows identical (1D problem), no transverse motion, volume fraction untouched
        assert np.array_equal(f["rho"][0], f["rho"][1])
        assert np.all(f["v"] == 0.0)
        np.testing.assert_allclose(f["q5"], 0.5, rtol=0, atol=1e-14)
    errs = np.array(errs)
    assert errs[2, 0] < 6e-3 and errs[2, 2] < 5e-3 and errs[2, 1] < 8e-3
    # convergence order ~ 0.8-1 for a solution with discontinuities
    assert np.all(errs[2] < 0.62 * errs[1]) and np.all(errs[1] < 0.62 * errs[0])


def test_sod_plateau_values(O):
    eos = dict(inputs.EOS, A=0.0, B=0.0, C=2.0, D=3.0, Gamma2=0.4, rho02=1.0)
    WL = [1.0, 1.0, 0.0, 0.0, 1.0, 0.5, 1.0]
    WR = [0.125, 0.125, 0.0, 0.0, 0.1, 0.5, 1.0]
    x, f, _ = _run_tube(O, eos, WL, WR, 0.5, 400, 0.2)
    ps, us = RX.star((1.0, 0.0, 1.0, 1.4, 0.0), (0.125, 0.0, 0.1, 1.4, 0.0))   # 0.30313, 0.92745
    m = (x > 0.60) & (x < 0.66)     # between tail of the fan and the contact
    assert np.allclose(f["p"][0][m], ps, rtol=2e-3) and np.allclose(f["u"][0][m], us, rtol=2e-3)
    m = (x > 0.72) & (x < 0.82)     # between contact and shock
    assert np.allclose(f["p"][0][m], ps, rtol=2e-3) and np.allclose(f["rho"][0][m], 0.26557, rtol=3e-3)


@pytest.mark.parametrize("limiter", [0, 1])
def test_water_air_shock_tube_against_exact_stiffened_gas_solution(O, limiter):
    # water: gamma 4.4, p_inf 6e8, rho 1000, p 1e9 | air: gamma 1.4, rho 50, p 1e5; interface at 0.7, t = 229 us
    pinf, gw = 6.0e8, 4.4
    eos = dict(inputs.EOS, gamma1=1.4, A=0.0, B=pinf, C=0.0, D=0.0, Gamma2=gw - 1.0, rho02=1000.0, z_min=1e-6)
    zm = 1e-6
    WL = [50.0, 1000.0, 0.0, 0.0, 1.0e9, zm, 1.0]
    WR = [50.0, 1000.0, 0.0, 0.0, 1.0e5, 1 - zm, 1.0]
    t_end = 229e-6
    left, right = (1000.0, 0.0, 1.0e9, gw, pinf), (50.0, 0.0, 1.0e5, 1.4, 0.0)
    errs = []
    for n in (200, 400):
        x, f, o = _run_tube(O, eos, WL, WR, 0.7, n, t_end, limiter=limiter)
        rho, u, p, isl = RX.sample(left, right, (x - 0.7) / t_end)
        errs.append((_l1(f["rho"][0], rho), np.mean(np.abs(f["u"][0] - u)) / np.max(u), _l1(f["p"][0], p)))
        # volume fraction follows the contact: total water volume changes only by compression-free advection
        xc = 0.7 + RX.star(left, right)[1] * t_end
        z2_int = np.sum(1.0 - f["q5"][0]) / n
        assert z2_int == pytest.approx(xc, abs=2.5 / n)
    errs = np.array(errs)
    print(errs)
    assert errs[1, 0] < 0.015 and errs[1, 1] < 0.02 and errs[1, 2] < 0.015
    assert np.all(errs[1] < 0.7 * errs[0])
    # star state on the plateau between rarefaction tail and contact
    ps, us = RX.star(left, right)
    m = (x > 0.55) & (x < 0.70 + us * t_end - 0.03)
    assert np.allclose(f["p"][0][m], ps, rtol=2e-2) and np.allclose(f["u"][0][m], us, rtol=2e-2)


def test_tube_along_y_equals_tube_along_x(O):
    # the y-sweep is the x-sweep with u <-> v: transposed problem gives the transposed answer bit for bit
    eos = dict(inputs.EOS, A=0.0, B=0.0, C=2.0, D=3.0, Gamma2=0.4, rho02=1.0)
    e = O.make_eos(eos)
    n = 64
    dx = 1.0 / n
    qL = O.prim_to_cons(e, [1.0, 1.0, 0.3, -0.2, 1.0, 0.3, 1.0])
    qR = O.prim_to_cons(e, [0.125, 0.125, 0.0, 0.1, 0.1, 0.6, 1.0])
    x = (np.arange(n) + 0.5) * dx
    qx = np.empty((7, 4, n))
    for k in range(7):
        qx[k] = np.where(x < 0.5, qL[k], qR[k])[None, :]
    gx = dict(nx=n, ny=4, dx=dx, dy=dx, bc_xlo=0, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=0)
    gy = dict(nx=4, ny=n, dx=dx, dy=dx, bc_xlo=1, bc_xhi=1, bc_ylo=0, bc_yhi=0, cfl=0.4, limiter=0)
    ox, oy = O.Oracle(gx, eos, KIN_OFF), O.Oracle(gy, eos, KIN_OFF)
    ox.init_fields(list(qx))
    qy = np.transpose(qx, (0, 2, 1)).copy()
    qy[[2, 3]] = qy[[3, 2]]
    oy.init_fields(list(qy))
    for _ in range(20):
        ox.sweep(0, 0.2 * dx)
        oy.sweep(1, 0.2 * dx)
    sx, sy = ox.state(), oy.state()
    perm = [0, 1, 3, 2, 4, 5, 6]
    for k in range(7):
        assert np.array_equal(sx[k], sy[perm[k]].T)
