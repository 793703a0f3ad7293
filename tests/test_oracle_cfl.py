"""Pins of the oracle's CFL step (a7, reading R11: dt = CFL min(dx,dy) / max_cells(max(|u|,|v|) + c)) and of everything
that depends on the cell shape (dt/dx vs dt/dy in the sweeps, dx*dy in Eq. 12), on grids with dx != dy.

The expected values are typed out here from closed forms, never taken from the oracle:
  * ideal gas in both phases (Cochran-Chan with A = B = 0, Gamma2 = gamma - 1): c = sqrt(gamma p / rho), textbook;
  * ambient nitromethane (Tables I-II): x = rho2/rho02 = 1, so Eq. 3 gives p_ref = A - B and
    rho2 c2^2 = A C - B D + (Gamma2 + 1)(p0 - (A - B))  ->  c = 1647.87 m/s;
  * Sod's tube along y on a grid with dx != dy against the exact Riemann solution (tests/riemann_exact.py).
"""
import math

import numpy as np
import pytest

import riemann_exact as RX
from paper_1905_05727_b200 import inputs

KIN_OFF = dict(inputs.KIN, reactive=0)
IDEAL = dict(inputs.EOS, A=0.0, B=0.0, C=2.0, D=3.0, Gamma2=0.4, rho02=1.0, z_min=1e-6)      # both phases gamma = 1.4


def _grid(nx, ny, dx, dy, bcx=(0, 0), bcy=(0, 0), cfl=0.4):
    return dict(nx=nx, ny=ny, dx=dx, dy=dy, bc_xlo=bcx[0], bc_xhi=bcx[1], bc_ylo=bcy[0], bc_yhi=bcy[1], cfl=cfl, limiter=0)


def _state(O, eos, W):
    """W[ny][nx] of primitive 7-vectors -> list of 7 conserved planes"""
    e = O.make_eos(eos)
    ny, nx = len(W), len(W[0])
    q = np.empty((7, ny, nx))
    for j in range(ny):
        for i in range(nx):
            q[:, j, i] = O.prim_to_cons(e, np.array(W[j][i], dtype=np.float64))
    return list(q)


# the four cells of the hand-built 2x2 state: (rho (both phases), u, v, p, z1); c = sqrt(1.4 p / rho) typed out below
# (every c is above the 1 m/s floor of R10; the floor has its own case below)
CELLS = [(1.0, 3.0, 0.5, 1.0, 0.3),        # c = sqrt(1.4)        = 1.1832159566199232, |u| + c = 4.183215956619923
         (0.5, -0.25, 1.0, 2.0, 0.6),      # c = sqrt(5.6)        = 2.3664319132398464, |v| + c = 3.366431913239846
         (2.0, 0.0, 0.0, 8.0, 0.5),        # c = sqrt(5.6)        = 2.3664319132398464
         (4.0, 1.0, -1.5, 7.0, 0.9)]       # c = sqrt(2.45)       = 1.5652475842498528, |v| + c = 3.0652475842498528
SPEEDS = [4.183215956619923, 3.366431913239846, 2.3664319132398464, 3.0652475842498528]


@pytest.mark.parametrize("dx,dy", [(1e-3, 0.7e-3), (0.4e-3, 1e-3), (1e-3, 1e-3)])
@pytest.mark.parametrize("boost", [None, (0, "u", 5.0), (1, "v", -7.0), (2, "u", -6.0), (3, "v", 9.0)])
def test_cfl_dt_on_a_hand_built_state(O, dx, dy, boost):
    """every cell in turn carries the maximum, once through |u| and once through |v| (negative velocities included)"""
    cells = [list(c) for c in CELLS]
    speeds = list(SPEEDS)
    if boost is not None:
        k, comp, val = boost
        cells[k][1 if comp == "u" else 2] = val
        rho, u, v, p, _ = cells[k]
        speeds[k] = max(abs(u), abs(v)) + math.sqrt(1.4 * p / rho)
    W = [[[c[0], c[0], c[1], c[2], c[3], c[4], 1.0] for c in cells[0:2]], [[c[0], c[0], c[1], c[2], c[3], c[4], 1.0] for c in cells[2:4]]]
    o = O.Oracle(_grid(2, 2, dx, dy), IDEAL, KIN_OFF)
    o.init_fields(_state(O, IDEAL, W))
    expect = 0.4 * min(dx, dy) / max(speeds)
    assert o.cfl_dt() == pytest.approx(expect, rel=1e-13)
    assert o.diagnostics()["smax"] == pytest.approx(max(speeds), rel=1e-13)
    # what separates the plausible mistakes from this value: max(dx, dy) differs whenever dx != dy; "|u| only" differs in the
    # cases whose maximum sits in |v| (boost 1 and 3), "|(u, v)|" in every case with both components non-zero
    if dx != dy:
        assert abs(0.4 * max(dx, dy) / max(speeds) / expect - 1.0) > 0.3
    if boost is not None and boost[1] == "v":
        u_only = max(abs(c[1]) + math.sqrt(1.4 * c[3] / c[0]) for c in cells)
        assert u_only < 0.8 * max(speeds)


def test_cfl_dt_ambient_nitromethane_typed_out(O):
    """Eq. 2-3 at x = 1 (Table II): rho2 c2^2 = A C - B D + (Gamma2 + 1)(p0 - A + B)"""
    A, B, Cc, D, G2, rho0, p0 = 0.819e9, 1.51e9, 4.53, 1.42, 1.19, 1134.0, 1.0e5
    c2 = math.sqrt((A * Cc - B * D + (G2 + 1.0) * (p0 - A + B)) / rho0)
    assert c2 == pytest.approx(1647.87, abs=0.01)
    zm = inputs.EOS["z_min"]
    amb = [1.2, rho0, 0.0, 0.0, p0, zm, 1.0]
    mov = [1.2, rho0, 120.0, -2500.0, p0, zm, 1.0]
    o = O.Oracle(_grid(3, 2, 5e-6, 2e-6), inputs.EOS, KIN_OFF)
    o.init_fields(_state(O, inputs.EOS, [[amb, amb, amb], [amb, amb, mov]]))
    # z1 = 1e-6 of air changes the frozen mixture sound speed (R10) by less than 1e-2 relative
    # (rho c^2 = [z1 gamma1 p/Gamma1 + z2 rho2 c2^2/Gamma2]/xi: the air term is 3.5e5 * 1e-6 against 2.6e9)
    assert o.cfl_dt() == pytest.approx(0.4 * 2e-6 / (2500.0 + c2), rel=1e-2)
    assert o.cfl_dt() == pytest.approx(0.4 * 2e-6 / (2500.0 + o.read_field("c")[1, 2]), rel=1e-14)
    assert o.read_field("c")[0, 0] == pytest.approx(c2, rel=1e-2)


def test_cfl_dt_uses_the_floored_sound_speed(O):
    """R10: c >= 1 m/s.  A cold, dense ideal-gas cell with sqrt(gamma p / rho) = 0.0374 must count as |u| + 1."""
    W = [[[1.0, 1.0, 2.0, 0.0, 1e-3, 0.5, 1.0], [1.0, 1.0, 0.0, -2.0, 1e-3, 0.5, 1.0]]]
    o = O.Oracle(_grid(2, 1, 1e-3, 2e-3), IDEAL, KIN_OFF)
    o.init_fields(_state(O, IDEAL, W))
    assert o.cfl_dt() == pytest.approx(0.4 * 1e-3 / 3.0, rel=1e-13)


def test_cfl_dt_ignores_ghost_cells_and_sees_every_cell(O):
    """the maximum may sit in any cell, including the last row / column; stale ghosts (a previous sweep's) do not count"""
    nx, ny = 5, 4
    base = [1.0, 1.0, 0.1, 0.1, 1.0, 0.5, 1.0]
    for (jj, ii) in [(0, 0), (ny - 1, nx - 1), (0, nx - 1), (ny - 1, 0), (2, 3)]:
        W = [[list(base) for _ in range(nx)] for _ in range(ny)]
        W[jj][ii][3] = -4.0
        o = O.Oracle(_grid(nx, ny, 2e-3, 1e-3), IDEAL, KIN_OFF)
        o.init_fields(_state(O, IDEAL, W))
        assert o.cfl_dt() == pytest.approx(0.4 * 1e-3 / (4.0 + math.sqrt(1.4)), rel=1e-13)


@pytest.mark.parametrize("ratio", [0.5, 3.0])
def test_sod_tube_along_y_on_a_non_square_grid(O, ratio):
    """dy = 1/n, dx = ratio * dy: the y-sweep must use dt/dy and the step min(dx, dy); with dt/dx instead every wave would
    travel 1/ratio times too far and the comparison with the exact solution would fail by tens of per cent"""
    n = 200
    dy = 1.0 / n
    dx = ratio * dy
    g = _grid(3, n, dx, dy, bcx=(1, 1), bcy=(0, 0))
    o = O.Oracle(g, IDEAL, KIN_OFF)
    y = (np.arange(n) + 0.5) * dy
    WL, WR = [1.0, 1.0, 0.0, 0.0, 1.0, 0.5, 1.0], [0.125, 0.125, 0.0, 0.0, 0.1, 0.5, 1.0]
    o.init_fields(_state(O, IDEAL, [[WL if yy < 0.5 else WR for _ in range(3)] for yy in y]))
    t_end, nsteps = 0.2, 0
    while True:
        dt, t = o.cfl_dt(), o.diagnostics()["t"]
        smax = o.diagnostics()["smax"]
        assert dt == pytest.approx(0.4 * min(dx, dy) / smax, rel=1e-13)
        if t + dt >= t_end:
            o.step_dt(1, t_end - t)
            break
        o.step_dt(1, dt)
        nsteps += 1
    rho, v, p, _ = RX.sample((1.0, 0.0, 1.0, 1.4, 0.0), (0.125, 0.0, 0.1, 1.4, 0.0), (y - 0.5) / t_end)
    f = {k: o.read_field(k) for k in ("rho", "u", "v", "p")}
    assert np.mean(np.abs(f["rho"][:, 1] - rho)) / np.mean(rho) < 1.2e-2
    assert np.mean(np.abs(f["p"][:, 1] - p)) / np.mean(p) < 1.0e-2
    assert np.mean(np.abs(f["v"][:, 1] - v)) < 1.6e-2
    assert np.all(f["u"] == 0.0) and np.array_equal(f["rho"][:, 0], f["rho"][:, 2])
    # the shock sits where the exact solution puts it: first row from the top with p > 0.2 within 2 cells of 0.5 + 1.75216 t
    front = y[np.max(np.flatnonzero(f["p"][:, 1] > 0.2))]
    assert front == pytest.approx(0.5 + 1.7521557320301779 * t_end, abs=2.5 * dy)
    # with dx < dy the step is limited by dx: about 1/ratio times as many steps
    if ratio < 1.0:
        assert nsteps > 1.8 * 0.2 / (0.4 * dy / 2.2)


def test_diagnostics_use_the_cell_area(O):
    """Eq. 12: M2r = sum q6 dx dy; conservation sums likewise.  Uniform ambient NM on a 7 x 3 grid, dx != dy."""
    nx, ny, dx, dy = 7, 3, 3e-6, 5e-6
    zm = inputs.EOS["z_min"]
    amb = [1.2, 1134.0, 10.0, -20.0, 1.0e5, zm, 1.0]
    o = O.Oracle(_grid(nx, ny, dx, dy), inputs.EOS, KIN_OFF)
    o.init_fields(_state(O, inputs.EOS, [[amb] * nx for _ in range(ny)]))
    d = o.diagnostics()
    area = nx * dx * ny * dy
    assert d["M2r"] == pytest.approx(1134.0 * (1 - zm) * area, rel=1e-13) and d["M2tot0"] == pytest.approx(d["M2r"], rel=1e-14)
    assert d["mass1"] == pytest.approx(1.2 * zm * area, rel=1e-13)
    rho = 1.2 * zm + 1134.0 * (1 - zm)
    assert d["momx"] == pytest.approx(rho * 10.0 * area, rel=1e-13) and d["momy"] == pytest.approx(-rho * 20.0 * area, rel=1e-13)
