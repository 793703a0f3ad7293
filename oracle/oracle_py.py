"""ctypes binding of liboracle.so -- TEST INFRASTRUCTURE (see nmsdt_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It mirrors the structs of nmsdt_oracle.h; it shares nothing with paper_1905_05727_b200.
"""
import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)
import build as _build  # noqa: E402  (oracle/build.py)

BC_TRANSMISSIVE, BC_PERIODIC, BC_REFLECTIVE, BC_INFLOW_FIXED = 0, 1, 2, 3
LIM_MINMOD, LIM_MC = 0, 1
FIELD = {"q0": 0, "q1": 1, "q2": 2, "q3": 3, "q4": 4, "q5": 5, "q6": 6, "p": 16, "T2": 17, "rho": 18, "u": 19,
         "v": 20, "lambda": 21, "progress": 22, "rho2": 23, "c": 24, "T1": 25, "rho1": 26}


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("dx", C.c_double), ("dy", C.c_double),
                ("bc_xlo", C.c_int), ("bc_xhi", C.c_int), ("bc_ylo", C.c_int), ("bc_yhi", C.c_int),
                ("cfl", C.c_double), ("limiter", C.c_int)]


class Eos(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("gamma1", "cv1", "Gamma2", "A", "B", "C", "D", "rho02", "cv2", "Tref2", "z_min")]


class Kin(C.Structure):
    _fields_ = [("Ta", C.c_double), ("Cpre", C.c_double), ("Q", C.c_double), ("reactive", C.c_int),
                ("max_substeps", C.c_int), ("substep_theta", C.c_double)]


class Cavity(C.Structure):
    _fields_ = [("x", C.c_double), ("y", C.c_double), ("r", C.c_double)]


class Init(C.Structure):
    _fields_ = [("p_shock", C.c_double), ("shock_cells", C.c_int), ("p0", C.c_double), ("rho1_0", C.c_double),
                ("rho2_0", C.c_double), ("interface_width", C.c_double), ("cav", C.POINTER(Cavity)),
                ("ncav", C.c_int), ("seed", C.c_ulonglong), ("phi", C.c_double), ("dmin", C.c_double),
                ("dmax", C.c_double), ("min_gap", C.c_double), ("x_lo", C.c_int), ("x_hi", C.c_int),
                ("lattice", C.c_int), ("lattice_d", C.c_double), ("lattice_spacing", C.c_double)]


class Diag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_longlong), ("dt_last", C.c_double), ("smax", C.c_double),
                ("M2r", C.c_double), ("M2tot0", C.c_double), ("burned_mass", C.c_double), ("rate_inst", C.c_double),
                ("mass1", C.c_double), ("mass2", C.c_double), ("momx", C.c_double), ("momy", C.c_double),
                ("energy", C.c_double), ("bad_state", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        for name, res, args in [
            ("orc_pref2", C.c_double, [C.POINTER(Eos), C.c_double]),
            ("orc_eref2", C.c_double, [C.POINTER(Eos), C.c_double]),
            ("orc_e2", C.c_double, [C.POINTER(Eos), C.c_double, C.c_double]),
            ("orc_T2", C.c_double, [C.POINTER(Eos), C.c_double, C.c_double]),
            ("orc_T1", C.c_double, [C.POINTER(Eos), C.c_double, C.c_double]),
            ("orc_mix_rhoe", C.c_double, [C.POINTER(Eos), C.c_double, C.c_double, C.c_double]),
            ("orc_mix_p", C.c_double, [C.POINTER(Eos), C.c_double, C.c_double, C.c_double]),
            ("orc_mix_rhoc2", C.c_double, [C.POINTER(Eos), C.c_double, C.c_double, C.c_double]),
            ("orc_limiter", C.c_double, [C.c_int, C.c_double, C.c_double]),
            ("orc_cons_to_prim", None, [C.POINTER(Eos), dp, dp, dp, dp]),
            ("orc_prim_to_cons", None, [C.POINTER(Eos), dp, dp]),
            ("orc_hllc", None, [C.POINTER(Eos), dp, dp, dp, dp]),
            ("orc_source_cell", C.c_int, [C.POINTER(Eos), C.POINTER(Kin), dp, C.c_double]),
            ("orc_hugoniot", C.c_int, [C.POINTER(Eos), C.c_double, C.c_double, C.c_double, C.c_double, dp]),
            ("orc_gen_cavities", C.c_int, [C.c_ulonglong, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int,
                                           C.c_int, C.c_int, C.c_int, C.POINTER(Cavity), C.c_int]),
            ("orc_create", C.c_int, [C.POINTER(Grid), C.POINTER(Eos), C.POINTER(Kin), C.POINTER(C.c_void_p)]),
            ("orc_destroy", None, [C.c_void_p]),
            ("orc_set_threads", None, [C.c_void_p, C.c_int]),
            ("orc_init", C.c_int, [C.c_void_p, C.POINTER(Init)]),
            ("orc_init_fields", C.c_int, [C.c_void_p, C.POINTER(dp)]),
            ("orc_cfl_dt", C.c_int, [C.c_void_p, dp]),
            ("orc_step", C.c_int, [C.c_void_p, C.c_int]),
            ("orc_step_dt", C.c_int, [C.c_void_p, C.c_int, C.c_double]),
            ("orc_diagnostics", C.c_int, [C.c_void_p, C.POINTER(Diag)]),
            ("orc_read_field", C.c_int, [C.c_void_p, C.c_int, dp]),
            ("orc_profiles", C.c_int, [C.c_void_p, C.c_double, dp, dp, dp, dp]),
            ("orc_qdot_pdf", C.c_int, [C.c_void_p, C.c_double, C.c_double, C.c_int, dp, C.POINTER(C.c_longlong)]),
            ("orc_shock_kinematics", C.c_int, [dp, dp, C.c_int, C.c_double, dp, dp]),
            ("orc_get_cavities", C.c_int, [C.c_void_p, C.POINTER(Cavity), C.c_int, C.POINTER(C.c_int)]),
            ("orc_fallback_count", C.c_longlong, [C.c_void_p]),
            ("orc_halo", C.c_int, [C.c_void_p, C.c_int]),
            ("orc_sweep", C.c_int, [C.c_void_p, C.c_int, C.c_double]),
            ("orc_source", C.c_int, [C.c_void_p, C.c_double]),
        ]:
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _fill(struct, d):
    for k, v in d.items():
        setattr(struct, k, v)
    return struct


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_eos(d):
    return _fill(Eos(), d)


def make_kin(d):
    return _fill(Kin(), d)


def make_init(d):
    """dict -> (Init struct, keep-alive list)."""
    d = dict(d)
    keep = []
    ini = Init()
    cav = d.pop("cavities", None)
    _fill(ini, d)
    if cav is not None and len(cav) > 0:
        arr = (Cavity * len(cav))(*[Cavity(float(c[0]), float(c[1]), float(c[2])) for c in cav])
        keep.append(arr)
        ini.cav = C.cast(arr, C.POINTER(Cavity))
        ini.ncav = len(cav)
    return ini, keep


class Oracle:
    """One oracle simulation. grid/eos/kin/init are plain dicts (see paper_1905_05727_b200.inputs)."""

    def __init__(self, grid, eos, kin, threads=1):
        self.L = lib()
        self.grid = _fill(Grid(), grid)
        self.eos = make_eos(eos)
        self.kin = make_kin(kin)
        self.h = C.c_void_p()
        rc = self.L.orc_create(C.byref(self.grid), C.byref(self.eos), C.byref(self.kin), C.byref(self.h))
        if rc != 0:
            raise ValueError("orc_create failed: %d" % rc)
        self.L.orc_set_threads(self.h, int(threads))
        self.nx, self.ny = self.grid.nx, self.grid.ny

    def close(self):
        if self.h:
            self.L.orc_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc != 0:
            raise RuntimeError("%s failed: %d" % (what, rc))

    def init(self, init):
        ini, keep = make_init(init)
        self._chk(self.L.orc_init(self.h, C.byref(ini)), "orc_init")

    def init_fields(self, q):
        q = [np.ascontiguousarray(a, dtype=np.float64).reshape(self.ny, self.nx) for a in q]
        ptrs = (C.POINTER(C.c_double) * 7)(*[_dp(a) for a in q])
        self._chk(self.L.orc_init_fields(self.h, ptrs), "orc_init_fields")

    def cfl_dt(self):
        dt = C.c_double()
        self._chk(self.L.orc_cfl_dt(self.h, C.byref(dt)), "orc_cfl_dt")
        return dt.value

    def step(self, n=1):
        self._chk(self.L.orc_step(self.h, int(n)), "orc_step")

    def step_dt(self, n, dt):
        self._chk(self.L.orc_step_dt(self.h, int(n), float(dt)), "orc_step_dt")

    def halo(self, d):
        self._chk(self.L.orc_halo(self.h, int(d)), "orc_halo")

    def sweep(self, d, dt):
        self._chk(self.L.orc_sweep(self.h, int(d), float(dt)), "orc_sweep")

    def source(self, tau):
        self._chk(self.L.orc_source(self.h, float(tau)), "orc_source")

    def diagnostics(self):
        d = Diag()
        self._chk(self.L.orc_diagnostics(self.h, C.byref(d)), "orc_diagnostics")
        return {n: getattr(d, n) for n, _ in Diag._fields_}

    def read_field(self, fid):
        if isinstance(fid, str):
            fid = FIELD[fid]
        out = np.empty((self.ny, self.nx), dtype=np.float64)
        self._chk(self.L.orc_read_field(self.h, int(fid), _dp(out)), "orc_read_field")
        return out

    def profiles(self, p_front):
        """Eq. 9-11 and the Appendix C front position: (pbar[nx], rhobar[nx], ubar[nx], x_s)"""
        pb, rb, ub = (np.empty(self.nx, dtype=np.float64) for _ in range(3))
        xs = C.c_double()
        self._chk(self.L.orc_profiles(self.h, float(p_front), _dp(pb), _dp(rb), _dp(ub), C.byref(xs)), "orc_profiles")
        return pb, rb, ub, xs.value

    def qdot_pdf(self, n_lo=2.0, dn=0.02, nbins=400):
        """Eq. 14-16: (mass[nbins], count[nbins])"""
        m = np.empty(nbins, dtype=np.float64)
        c = np.empty(nbins, dtype=np.int64)
        self._chk(self.L.orc_qdot_pdf(self.h, float(n_lo), float(dn), int(nbins), _dp(m),
                                      c.ctypes.data_as(C.POINTER(C.c_longlong))), "orc_qdot_pdf")
        return m, c

    def state(self):
        return [self.read_field(k) for k in range(7)]

    def cavities(self):
        n = C.c_int()
        self.L.orc_get_cavities(self.h, None, 0, C.byref(n))
        arr = (Cavity * max(n.value, 1))()
        self.L.orc_get_cavities(self.h, arr, n.value, C.byref(n))
        return np.array([[arr[i].x, arr[i].y, arr[i].r] for i in range(n.value)], dtype=np.float64).reshape(-1, 3)

    def fallback_count(self):
        return int(self.L.orc_fallback_count(self.h))


# ---- pointwise helpers (numpy scalars in, python floats out) ------------------------------------------

def cons_to_prim(eos, q):
    q = np.ascontiguousarray(q, dtype=np.float64)
    W = np.empty(7)
    c = C.c_double()
    T2 = C.c_double()
    lib().orc_cons_to_prim(C.byref(eos), _dp(q), _dp(W), C.byref(c), C.byref(T2))
    return W, c.value, T2.value


def prim_to_cons(eos, W):
    W = np.ascontiguousarray(W, dtype=np.float64)
    q = np.empty(7)
    lib().orc_prim_to_cons(C.byref(eos), _dp(W), _dp(q))
    return q


def hllc(eos, WL, WR):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.empty(7)
    u = C.c_double()
    lib().orc_hllc(C.byref(eos), _dp(WL), _dp(WR), _dp(F), C.byref(u))
    return F, u.value


def source_cell(eos, kin, q, tau):
    q = np.array(q, dtype=np.float64)
    n = lib().orc_source_cell(C.byref(eos), C.byref(kin), _dp(q), float(tau))
    return q, n


def hugoniot(eos, p0, rho1_0, rho2_0, ps):
    out = np.empty(5)
    rc = lib().orc_hugoniot(C.byref(eos), p0, rho1_0, rho2_0, ps, _dp(out))
    if rc != 0:
        raise RuntimeError("orc_hugoniot failed")
    return dict(rho_s=out[0], U_s=out[1], u_p=out[2], T2_s=out[3], rho1_s=out[4])


def gen_cavities(seed, phi, dmin, dmax, min_gap, x_lo, x_hi, ny, periodic_y, cap=1 << 20):
    arr = (Cavity * cap)()
    n = lib().orc_gen_cavities(seed, phi, dmin, dmax, min_gap, x_lo, x_hi, ny, int(periodic_y), arr, cap)
    if n < 0:
        raise RuntimeError("orc_gen_cavities failed")
    return np.array([[arr[i].x, arr[i].y, arr[i].r] for i in range(n)], dtype=np.float64).reshape(-1, 3)


def shock_kinematics(t, xs, dtau):
    """Eq. C1-C2: (u_s[n], a_s[n]), NaN where the window leaves the sampled interval"""
    t = np.ascontiguousarray(t, dtype=np.float64)
    xs = np.ascontiguousarray(xs, dtype=np.float64)
    us, a = np.empty_like(t), np.empty_like(t)
    rc = lib().orc_shock_kinematics(_dp(t), _dp(xs), int(t.size), float(dtau), _dp(us), _dp(a))
    if rc != 0:
        raise RuntimeError("orc_shock_kinematics failed: %d" % rc)
    return us, a
