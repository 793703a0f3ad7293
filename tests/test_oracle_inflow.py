"""Pin of the oracle's fixed-inflow boundary (orc_halo case ORC_BC_INFLOW_FIXED and the capture in finish_init; reading R12 of
DESIGN.md / SURVEY A12 for PAPER.md P:129 "inflow (transmissive)": the two ghost columns at x-lo hold, for the whole run, the
state column 0 had when the run was initialised).

The pin needs no access to fluxes.  Both phases are the same ideal gas (A = B = 0 as in the Sod pin) and the flow is supersonic
to the right everywhere (u > c), so that
  * the two ghost cells of a row are equal -> the limited slope in the ghost cell next to the boundary is 0 for either limiter,
    its face state is the ghost state itself, untouched by the Hancock predictor;
  * HLLC with all waves running to the right returns the physical flux of its left state (`test_hllc_is_consistent_and_upwinds`);
  * at x-hi (transmissive) both face states are the last cell: HLLC(W, W) = F(W).
One x-sweep then changes the row sums by exactly  dt/dx (F(W_ghost(j)) - F(W_last(j)))  for the conserved components, with both
fluxes TYPED OUT below from primitive values.  The column-0 state is given a y-variation and the interior differs from it, so a
few full steps move the current column 0 well away from the captured one: the budget holds with the captured state and fails by
orders of magnitude with the current one -- and the other way round for the transmissive rule on the same data.  A capture
taken at the wrong time or from another column, ghosts filled from the current column, or a second ghost column left unfilled fail
this test (tried by hand on mutated copies of the oracle)."""
import numpy as np
import pytest

from paper_1905_05727_b200 import inputs

KIN_OFF = dict(inputs.KIN, reactive=0)
GAMMA = 1.4
EOS_IDEAL = dict(inputs.EOS, gamma1=GAMMA, A=0.0, B=0.0, C=2.0, D=3.0, Gamma2=GAMMA - 1.0, rho02=1.0, z_min=1e-6)
NX, NY, DX = 48, 6, 1.0 / 48


def _physical_flux(W):
    """x-flux of the conserved components (q0, q1, q2, q3, q4, q6) of Eq. 1 for the ideal-gas mixture, from
    primitives W = (rho1, rho2, u, v, p, z1, lambda), arrays over rows"""
    r1, r2, u, v, p, z1, lam = W
    rho = z1 * r1 + (1.0 - z1) * r2
    rhoE = p / (GAMMA - 1.0) + 0.5 * rho * (u * u + v * v)          # both phases: rho e = p / (gamma - 1)
    return np.array([z1 * r1 * u, (1.0 - z1) * r2 * u, rho * u * u + p, rho * u * v, (rhoE + p) * u, (1.0 - z1) * r2 * lam * u])


def _prims_of_column(o, i):
    f = {k: o.read_field(k)[:, i] for k in ("rho1", "rho2", "u", "v", "p", "q5", "lambda")}
    return np.array([f["rho1"], f["rho2"], f["u"], f["v"], f["p"], f["q5"], f["lambda"]])


def _initial_prims():
    j = (np.arange(NY) + 0.5) / NY
    i = (np.arange(NX) + 0.5) / NX
    W = np.empty((7, NY, NX))
    # column 0: varies along y only, Mach 2.3-3.2
    col = np.array([1.0 + 0.2 * np.sin(2 * np.pi * j), 1.3 + 0.1 * np.cos(2 * np.pi * j), 3.2 + 0.4 * np.cos(2 * np.pi * j),
                    0.6 * np.sin(2 * np.pi * j), 1.0 + 0.15 * np.sin(4 * np.pi * j), 0.5 + 0.0 * j, 0.9 - 0.3 * j])
    # interior: a different, x-dependent state (still supersonic), so that column 0 changes from the first step on
    bump = np.exp(-((i - 0.25) / 0.12) ** 2)[None, :]
    for k in range(7):
        W[k] = col[k][:, None]
    W[0] *= 1.0 + 0.5 * bump
    W[1] *= 1.0 + 0.4 * bump
    W[2] += 0.5 * bump
    W[4] *= 1.0 + 0.8 * bump
    W[6] *= 1.0 - 0.5 * bump
    W[:, :, 0] = col
    return W, col


def _run(O, bc_xlo, limiter):
    g = dict(nx=NX, ny=NY, dx=DX, dy=DX, bc_xlo=bc_xlo, bc_xhi=0, bc_ylo=1, bc_yhi=1, cfl=0.4, limiter=limiter)
    o = O.Oracle(g, EOS_IDEAL, KIN_OFF)
    e = O.make_eos(EOS_IDEAL)
    W, col = _initial_prims()
    q = np.empty_like(W)
    for j in range(NY):
        for i in range(NX):
            q[:, j, i] = O.prim_to_cons(e, W[:, j, i])
    # the typed-out energy agrees with the oracle's own conversion (pinned elsewhere): the flux below speaks of the same state
    rho = W[5] * W[0] + (1 - W[5]) * W[1]
    np.testing.assert_allclose(q[4], W[4] / (GAMMA - 1.0) + 0.5 * rho * (W[2] ** 2 + W[3] ** 2), rtol=1e-14)
    o.init_fields(list(q))
    o.step(4)                                                        # full steps (x and y sweeps): column 0 leaves its initial state
    c = np.sqrt(GAMMA * o.read_field("p") / o.read_field("rho"))
    assert np.all(o.read_field("u") - c > 0.5), "the pin needs supersonic flow to the right everywhere"
    before = [a.copy() for a in o.state()]
    cur0, last = _prims_of_column(o, 0), _prims_of_column(o, NX - 1)
    dt = 0.8 * o.cfl_dt()
    o.sweep(0, dt)
    after = o.state()
    assert o.fallback_count() == 0
    change = np.array([(after[k] - before[k]).sum(axis=1) for k in (0, 1, 2, 3, 4, 6)])       # per row
    return change, dt / DX, col, cur0, last


@pytest.mark.parametrize("limiter", [0, 1])
def test_fixed_inflow_ghosts_hold_the_column_captured_at_init(O, limiter):
    change, dtdx, captured, cur0, last = _run(O, 3, limiter)
    # the steps have moved column 0 away from the captured state (otherwise the test could not tell the two apart)
    assert np.max(np.abs(cur0[4] / captured[4] - 1.0)) > 0.02 and np.max(np.abs(cur0[0] / captured[0] - 1.0)) > 0.02
    want = dtdx * (_physical_flux(captured) - _physical_flux(last))
    scale = dtdx * np.abs(_physical_flux(captured)).max(axis=1, keepdims=True)
    assert np.max(np.abs(change - want) / scale) < 5e-13
    wrong = dtdx * (_physical_flux(cur0) - _physical_flux(last))                # ghost = current column 0 (the transmissive rule)
    assert np.max(np.abs(change - wrong) / scale) > 1e-3
    # every row carries its OWN captured state (a y-shift of the captured column is seen)
    shifted = dtdx * (_physical_flux(np.roll(captured, 1, axis=1)) - _physical_flux(last))
    assert np.max(np.abs(change - shifted) / scale) > 1e-3


def test_transmissive_inflow_on_the_same_data_uses_the_current_column(O):
    change, dtdx, captured, cur0, last = _run(O, 0, 0)
    scale = dtdx * np.abs(_physical_flux(cur0)).max(axis=1, keepdims=True)
    assert np.max(np.abs(change - dtdx * (_physical_flux(cur0) - _physical_flux(last))) / scale) < 5e-13
    assert np.max(np.abs(change - dtdx * (_physical_flux(captured) - _physical_flux(last))) / scale) > 1e-3
