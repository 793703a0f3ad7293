"""Seeded, synthetic workload recipes shared by the tests, bench.py and smoke().

This module holds none of the method's arithmetic on fields: only the constants the paper prints
(Tables I-III; ambient state P:141) and the grid / cavity-layout / boundary
parameters of the five BASELINE.json configs.
Both the CUDA library and the oracle turn these plain dicts into fields with their own code.
One formula of the paper does appear: `paper_case` uses Eq. 7 (delta_c = sqrt(pi d_c^2 / 4 phi))
to write the EXPLICIT cavity list of the regular array, which both sides then receive as a list;
the oracle's own Eq. 7 is pinned apart from it (tests/test_oracle_init.py).

The paper measures on no public dataset; these generated fields take the shapes of its three
scenarios (neat NM, regular cavity array, hundreds of random cavities) and stand in
for its production grids (24000x313, 24000x2000 at dx = 1 um; `paper_case`, config names
'P313' / 'P2000' for bench.py), which the parity tests do not run.
"""
import copy

BC_TRANSMISSIVE, BC_PERIODIC, BC_REFLECTIVE, BC_INFLOW_FIXED = 0, 1, 2, 3
LIM_MINMOD, LIM_MC = 0, 1

# Table I, Table II (garbled labels read as A = 0.819 GPa, D = 1.42, DESIGN R2),
# T_ref,2 = 0 K; z_min from BASELINE.json config 2.
EOS = dict(gamma1=1.4, cv1=718.0, Gamma2=1.19, A=0.819e9, B=1.51e9, C=4.53, D=1.42, rho02=1134.0, cv2=1714.0,
           Tref2=0.0, z_min=1e-6)
# Table III; sub-stepping rule DESIGN R13
KIN = dict(Ta=11350.0, Cpre=2.6e9, Q=4.46e6, reactive=1, max_substeps=64, substep_theta=0.1)
# ambient state
AMBIENT = dict(p0=1.0e5, rho1_0=1.2, rho2_0=1134.0)

_INIT0 = dict(p_shock=8.0e9, shock_cells=0, interface_width=2.0, ncav=0, seed=0, phi=0.0, dmin=0.0, dmax=0.0,
              min_gap=0.0, x_lo=0, x_hi=0, lattice=0, lattice_d=0.0, lattice_spacing=0.0, **AMBIENT)


def _grid(nx, ny, dx, bcx=(BC_TRANSMISSIVE, BC_TRANSMISSIVE), bcy=(BC_PERIODIC, BC_PERIODIC), cfl=0.4,
          limiter=LIM_MINMOD):
    return dict(nx=nx, ny=ny, dx=dx, dy=dx, bc_xlo=bcx[0], bc_xhi=bcx[1], bc_ylo=bcy[0], bc_yhi=bcy[1], cfl=cfl,
                limiter=limiter)


def config(name, p_shock=None, reactive=None, nx=None, ny=None, seed=None):
    """Return dict(grid, eos, kin, init, steps, name) for BASELINE.json config 'C1'..'C5', or for the paper's two production
    grids 'P313' / 'P2000'.

    nx/ny override the grid size (a crop with the same generator parameters; the cavity
    region keeps its x_lo and is clipped to the new nx)."""
    if name in ("P313", "P2000"):
        # the paper's own production grids at dx = 1 um, as bench.py workloads: 24000 x 313 (regular array,
        # phi = 8 %) and 24000 x 2000 (random cavities, phi = 5 %, seed 2019), 7.81 GPa; see paper_case
        cfg = paper_case("regular" if name == "P313" else "random", 1.0, p_shock=7.81e9 if p_shock is None else p_shock,
                         seed=2019 if seed is None else seed)
        cfg["name"], cfg["steps"] = name, 200
        if nx is not None:
            cfg["grid"]["nx"] = int(nx)
            cfg["init"]["x_hi"] = min(cfg["init"]["x_hi"], int(nx))
            cfg["init"]["cavities"] = [c for c in cfg["init"].get("cavities", []) if c[0] + c[2] < nx]
        if ny is not None:
            cfg["grid"]["ny"] = int(ny)
            cfg["init"]["cavities"] = [c for c in cfg["init"].get("cavities", []) if c[1] + c[2] < ny]
        if reactive is not None:
            cfg["kin"]["reactive"] = int(reactive)
        return cfg
    eos, kin, init = copy.deepcopy(EOS), copy.deepcopy(KIN), copy.deepcopy(_INIT0)
    dx24 = 100e-6 / 24.0       # 24 cells per 100 um cavity diameter (DESIGN R21)
    if name == "C1":           # single cavity, 256x128, transmissive everywhere
        grid = _grid(256, 128, 100e-6 / 32.0, bcy=(BC_TRANSMISSIVE, BC_TRANSMISSIVE))
        init.update(p_shock=9.0e9, shock_cells=32, cavities=[(96.0, 64.0, 16.0)])
        steps = 200
    elif name == "C2":         # neat NM strip
        grid = _grid(4096, 32, 5e-6)
        init.update(p_shock=9.4e9, shock_cells=100)
        steps = 2000
    elif name == "C3":         # regular cavity array
        grid = _grid(4096, 512, dx24)
        init.update(p_shock=8.0e9, shock_cells=120, lattice=1, lattice_d=24.0, lattice_spacing=64.0, x_lo=512,
                    x_hi=4096)
        steps = 2000
    elif name == "C4":         # hundreds of random cavities
        grid = _grid(8192, 1024, dx24)
        init.update(p_shock=8.0e9, shock_cells=120, seed=12345, phi=0.03, dmin=24.0, dmax=24.0, min_gap=4.0,
                    x_lo=1024, x_hi=8192)
        steps = 2000
    elif name == "C5":         # large random field for roofline scaling
        grid = _grid(32768, 4096, dx24)
        init.update(p_shock=8.0e9, shock_cells=120, seed=12345, phi=0.05, dmin=16.0, dmax=40.0, min_gap=4.0,
                    x_lo=1024, x_hi=32768)
        steps = 200
    else:
        raise ValueError("unknown config %r" % (name,))
    if nx is not None:
        grid["nx"] = int(nx)
        if init["x_hi"]:
            init["x_hi"] = min(init["x_hi"], int(nx))
            if name == "C3" or init["phi"] > 0:
                init["x_lo"] = min(init["x_lo"], max(int(nx) // 4, init["shock_cells"] + 8))
    if ny is not None:
        grid["ny"] = int(ny)
    if p_shock is not None:
        init["p_shock"] = float(p_shock)
    if reactive is not None:
        kin["reactive"] = int(reactive)
    if seed is not None:
        init["seed"] = int(seed)
    return dict(name=name, grid=grid, eos=eos, kin=kin, init=init, steps=steps)


def paper_case(case, dx_um=1.0, p_shock=7.81e9, phi=None, seed=2019, length_mm=24.0):
    """The paper's own scenarios (Sect. IV, Appendix A) at grid spacing dx_um (paper: 1 um; Tables IV-V also
    give 4 and 2 um): 'neat' (W arbitrary: 32 cells), 'regular' (one row of d_c = 100 um cavities, W = delta_c of Eq. 7,
    phi = 8 %), 'random' (W = 2 mm, centre spacing >= 2.5 d_c, phi = 5 % as in Table V or 8 % as in Sect. IV).
    Domain length 24 mm, shocked slab L_s = 0.5 mm, input shock 7.81 GPa, periodic top / bottom."""
    import math
    eos, kin, init = copy.deepcopy(EOS), copy.deepcopy(KIN), copy.deepcopy(_INIT0)
    dx = dx_um * 1e-6
    nx = int(round(length_mm * 1e-3 / dx))
    ls = int(round(0.5e-3 / dx))
    dc = 100e-6 / dx                                   # cavity diameter in cells
    init.update(p_shock=float(p_shock), shock_cells=ls)
    if case == "neat":
        ny = 32
    elif case == "regular":
        phi = 0.08 if phi is None else phi
        delta = math.sqrt(math.pi * dc * dc / (4.0 * phi))            # Eq. 7, in cells
        ny = int(round(delta))
        # one row of cavities on the axis of a strip of width ny ~ delta (periodic images at distance ny), spacing delta in x
        ncol = int((nx - ls) / delta)
        init.update(cavities=[(ls + 0.5 * delta + delta * i, 0.5 * ny, 0.5 * dc) for i in range(ncol)])
    elif case == "random":
        phi = 0.05 if phi is None else phi
        ny = int(round(2.0e-3 / dx))
        init.update(seed=int(seed), phi=float(phi), dmin=dc, dmax=dc, min_gap=1.5 * dc, x_lo=ls, x_hi=nx)
    else:
        raise ValueError("unknown paper case %r" % (case,))
    return dict(name="paper-%s-dx%g" % (case, dx_um), grid=_grid(nx, ny, dx), eos=eos, kin=kin, init=init, steps=0)
