"""Pins of the oracle's problem setup (O7, R15, R16, R20): cavity generator (Eq. 7-8),
tanh painting, shocked slab, ambient state, M2,tot."""
import numpy as np
import pytest

from paper_1905_05727_b200 import inputs


def _brute_force_min_gap(cav, ny, periodic):
    n = len(cav)
    best = np.inf
    for a in range(n):
        d = cav[a + 1:, :2] - cav[a, :2]
        if periodic:
            d[:, 1] = np.abs(d[:, 1])
            d[:, 1] = np.minimum(d[:, 1], ny - d[:, 1])
        if len(d):
            gap = np.sqrt((d ** 2).sum(1)) - cav[a + 1:, 2] - cav[a, 2]
            best = min(best, gap.min())
    return best


def test_eq7_spacing_and_eq8_count():
    g = {}
    import os
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            g[k.strip()] = float(v)
    phi, dc = 0.08, 100e-6
    assert np.sqrt(np.pi * dc ** 2 / (4 * phi)) == pytest.approx(g["delta_c_mm"] * 1e-3, rel=2e-3)   # Eq. 7
    assert 4 * phi * 24e-3 * 2e-3 / (np.pi * dc ** 2) == pytest.approx(489, abs=1)                      # Eq. 8 "hundreds"


@pytest.mark.parametrize("periodic", [1, 0])
def test_generator_is_nonoverlapping_seeded_and_reaches_the_target_fraction(O, periodic):
    ny, x_lo, x_hi, phi, gap = 1024, 1024, 8192, 0.03, 4.0
    cav = O.gen_cavities(12345, phi, 24.0, 24.0, gap, x_lo, x_hi, ny, periodic)
    n_eq8 = 4 * phi * (x_hi - x_lo) * ny / (np.pi * 24.0 ** 2)        # Eq. 8 in cell units
    assert len(cav) == int(np.ceil(n_eq8))                           # ~487 cavities ("hundreds", P:7)
    assert np.all(cav[:, 2] == 12.0)
    assert _brute_force_min_gap(cav, ny, periodic) >= gap
    assert cav[:, 0].min() - 12 >= x_lo and cav[:, 0].max() + 12 <= x_hi
    if not periodic:
        assert cav[:, 1].min() - 12 >= 0 and cav[:, 1].max() + 12 <= ny
    else:
        assert cav[:, 1].min() >= 0 and cav[:, 1].max() < ny
    # fixed point 1/256 cell
    assert np.all(cav * 256 == np.round(cav * 256))
    # seeded: same seed same list, other seed other list
    assert np.array_equal(cav, O.gen_cavities(12345, phi, 24.0, 24.0, gap, x_lo, x_hi, ny, periodic))
    other = O.gen_cavities(54321, phi, 24.0, 24.0, gap, x_lo, x_hi, ny, periodic)
    assert len(other) == len(cav) and not np.array_equal(other, cav)
    # uniform placement: quadrant counts within 5 sigma of a quarter each
    qx = cav[:, 0] > 0.5 * (x_lo + x_hi)
    qy = cav[:, 1] > 0.5 * ny
    for m in (qx & qy, qx & ~qy, ~qx & qy, ~qx & ~qy):
        assert abs(m.sum() - len(cav) / 4) < 5 * np.sqrt(len(cav) * 3 / 16)


def test_generator_diameter_range_and_paper_spacing_rule(O):
    # R16: paper's rule "minimum spacing 2.5 d_c" = surface gap 1.5 d_c
    cav = O.gen_cavities(7, 0.02, 16.0, 40.0, 1.5 * 16.0, 256, 4096, 512, 1)
    d = 2 * cav[:, 2]
    assert d.min() >= 16.0 and d.max() <= 40.0 and d.std() > 4.0
    assert _brute_force_min_gap(cav, 512, True) >= 24.0
    area = np.pi * (cav[:, 2] ** 2).sum()
    target = 0.02 * (4096 - 256) * 512
    assert area >= target and area - np.pi * cav[-1, 2] ** 2 < target     # stops at the first crossing


def test_c1_initial_fields(O, paper_eos):
    c = inputs.config("C1")
    o = O.Oracle(c["grid"], c["eos"], c["kin"])
    o.init(c["init"])
    z1, p, u, lam, rho2, rho1 = (o.read_field(k) for k in ("q5", "p", "u", "lambda", "rho2", "rho1"))
    h = O.hugoniot(paper_eos, 1e5, 1.2, 1134.0, 9e9)
    # shocked slab: Hugoniot state, lambda = 0, neat NM
    assert np.allclose(p[:, :32], 9e9, rtol=1e-9) and np.allclose(u[:, :32], h["u_p"], rtol=1e-12)
    assert np.all(lam[:, :32] == 0.0) and np.all(z1[:, :32] == 1e-6)
    assert np.allclose(rho2[:, :32], h["rho_s"], rtol=1e-12)
    # ambient
    assert np.allclose(p[:, 32:], 1e5, rtol=1e-6) and np.all(u[:, 32:] == 0.0) and np.all(lam[:, 32:] == 1.0)
    assert np.allclose(rho2[:, 32:], 1134.0, rtol=1e-12) and np.allclose(rho1[:, 32:], 1.2, rtol=1e-9)
    # cavity: tanh profile of half-width h = 1 cell around r = 16 at (96, 64) (R15)
    yy, xx = np.meshgrid(np.arange(128) + 0.5, np.arange(256) + 0.5, indexing="ij")
    d = np.sqrt((xx - 96.0) ** 2 + (yy - 64.0) ** 2)
    expect = 1e-6 + (1 - 2e-6) * 0.5 * (1 - np.tanh((d - 16.0) / 1.0))
    expect[:, :32] = 1e-6
    np.testing.assert_allclose(z1, expect, rtol=0, atol=1e-15)
    assert z1[64, 96] > 1 - 2e-6 and z1[0, 255] == 1e-6
    # area of a radial tanh profile: pi (R^2 + pi^2 h^2 / 12)
    assert (z1 - 1e-6).sum() == pytest.approx(np.pi * (16.0 ** 2 + np.pi ** 2 / 12), rel=1e-4)
    # M2,tot = rho2 (1 - phi) L W over the reactive region
    d0 = o.diagnostics()
    dx = c["grid"]["dx"]
    phi = np.pi * (16.0 ** 2 + np.pi ** 2 / 12) / ((256 - 32) * 128)
    assert d0["M2tot0"] == pytest.approx(1134.0 * (1 - phi) * (256 - 32) * 128 * dx * dx, rel=1e-4)
    assert d0["M2r"] == d0["M2tot0"] and d0["burned_mass"] == 0.0


def test_lattice_and_periodic_painting(O):
    c = inputs.config("C3", nx=512, ny=128)
    o = O.Oracle(c["grid"], c["eos"], c["kin"])
    o.init(c["init"])
    cav = o.cavities()
    # R20: centres x_lo + 32 + 64 i, 32 + 64 j
    x_lo = c["init"]["x_lo"]
    assert len(cav) == ((512 - x_lo) // 64) * 2
    assert set(cav[:, 1]) == {32.0, 96.0} and cav[:, 0].min() == x_lo + 32.0
    z1 = o.read_field("q5")
    assert z1[32, x_lo + 32] > 0.999 and z1[0, x_lo + 32] < 1e-5
    # periodic minimum image: a cavity centred on the y-boundary paints both edges symmetrically
    g = dict(c["grid"], nx=64, ny=64)
    ini = dict(c["init"], lattice=0, shock_cells=0, cavities=[(32.0, 0.0, 10.0)])
    o = O.Oracle(g, c["eos"], c["kin"])
    o.init(ini)
    z = o.read_field("q5")
    assert np.array_equal(z[:8], z[::-1][:8]) and z[0, 31] > 0.999 and z[32, 31] == 1e-6
    # the same cavity in a transmissive box is cut, not wrapped
    g2 = dict(g, bc_ylo=0, bc_yhi=0)
    o2 = O.Oracle(g2, c["eos"], c["kin"])
    o2.init(ini)
    z2 = o2.read_field("q5")
    assert z2[0, 31] > 0.999 and z2[63, 31] == 1e-6


def test_init_fields_clamps_the_volume_fraction(O):
    """R27: an explicit initial state is stored with q5 in [z_min, 1 - z_min] (the invariant O7 / O4.6 / O3 keep for every
    state of the scheme); values inside are stored bit for bit, the other six fields are never touched."""
    cfg = inputs.config("C2", nx=8, ny=4, reactive=0)
    zmin = cfg["eos"]["z_min"]
    o = O.Oracle(cfg["grid"], cfg["eos"], cfg["kin"])
    o.init(dict(cfg["init"], shock_cells=2))
    q = [a.copy() for a in o.state()]
    q[5][0, :] = [0.0, -0.25, 1.0, 1.5, zmin, 1.0 - zmin, 0.5 * zmin, 0.3]
    keep = [a.copy() for a in q]
    o.init_fields(q)
    got = o.state()
    assert np.array_equal(got[5][0], [zmin, zmin, 1.0 - zmin, 1.0 - zmin, zmin, 1.0 - zmin, zmin, 0.3])
    assert np.array_equal(got[5][1:], keep[5][1:])
    for k in (0, 1, 2, 3, 4, 6):
        assert np.array_equal(got[k], keep[k])
