"""Thin ctypes binding of libnmsdt.so (include/nmsdt.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch is used for device memory
(the workspace is a torch uint8 tensor lent to sim_create) and for the CUDA stream.  There is no CPU
fallback: importing works anywhere (so that symbol checks can run without a GPU), but creating a `Sim`
without the built library or without a CUDA device raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libnmsdt.so")

SIM_OK, SIM_ERR_ARG, SIM_ERR_CUDA, SIM_ERR_STATE, SIM_ERR_BAD = 0, -1, -2, -3, -4
VARIANT_UNFUSED, VARIANT_FUSED = 0, 1
FIELD = {"q0": 0, "q1": 1, "q2": 2, "q3": 3, "q4": 4, "q5": 5, "q6": 6, "p": 16, "T2": 17, "rho": 18, "u": 19,
         "v": 20, "lambda": 21, "progress": 22, "rho2": 23, "c": 24, "T1": 25, "rho1": 26}

# every symbol include/nmsdt.h declares (tests check that the library exports each one)
SYMBOLS = ["sim_workspace_bytes", "sim_create", "sim_destroy", "sim_last_error", "sim_init", "sim_init_fields",
           "sim_cfl_dt", "sim_step", "sim_step_dt", "sim_halo", "sim_sweep", "sim_source", "sim_diagnostics",
           "sim_read_field", "sim_get_cavities", "sim_cavity_stats", "sim_redo_count", "sim_set_variant", "sim_set_launch_mode", "sim_sweep_geometry", "sim_launch_count", "sim_device_layout",
           "sim_probe_fp64", "sim_probe_issue", "sim_probe_math", "sim_profile", "sim_kernel_time", "sim_profiles", "sim_qdot_pdf",
           "sim_qdot_pdf_noalloc",
           "sim_shock_kinematics", "sim_init_slab", "sim_slab_halo_bytes", "sim_slab_begin", "sim_slab_smax_ptr",
           "sim_slab_ctl", "sim_slab_pass_dir", "sim_slab_pass", "sim_slab_pack", "sim_slab_unpack", "sim_slab_info",
           "sim_slab_connect", "sim_slab_push", "sim_slab_ipc_export", "sim_slab_ipc_open", "sim_slab_ipc_close"]
BC_EXTERNAL = 4
KERNEL_KINDS = {"sweep_x": 0, "sweep_y": 1, "source": 2, "cfl": 3, "halo": 4}


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


class SlabPeer(C.Structure):
    _fields_ = [("plane0", C.c_void_p * 2), ("plane_stride", C.c_longlong), ("pitch", C.c_int), ("nx", C.c_int),
                ("ny", C.c_int)]


class NmsdtError(RuntimeError):
    def __init__(self, what, code, msg):
        super().__init__("%s failed (%d): %s" % (what, code, msg))
        self.code = code


_lib = None


def load_library():
    """Load libnmsdt.so (no CUDA call is made). Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libnmsdt.so is not built: run `python -m paper_1905_05727_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    dp, vp = C.POINTER(C.c_double), C.c_void_p
    sig = {
        "sim_workspace_bytes": (C.c_size_t, [C.POINTER(Grid)]),
        "sim_create": (C.c_int, [C.POINTER(Grid), C.POINTER(Eos), C.POINTER(Kin), vp, C.c_size_t, vp, C.POINTER(vp)]),
        "sim_destroy": (None, [vp]),
        "sim_last_error": (C.c_char_p, [vp]),
        "sim_init": (C.c_int, [vp, C.POINTER(Init)]),
        "sim_init_fields": (C.c_int, [vp, C.POINTER(dp)]),
        "sim_cfl_dt": (C.c_int, [vp, dp]),
        "sim_step": (C.c_int, [vp, C.c_int]),
        "sim_step_dt": (C.c_int, [vp, C.c_int, C.c_double]),
        "sim_halo": (C.c_int, [vp, C.c_int]),
        "sim_sweep": (C.c_int, [vp, C.c_int, C.c_double]),
        "sim_source": (C.c_int, [vp, C.c_double]),
        "sim_diagnostics": (C.c_int, [vp, C.POINTER(Diag)]),
        "sim_read_field": (C.c_int, [vp, C.c_int, dp]),
        "sim_get_cavities": (C.c_int, [vp, C.POINTER(Cavity), C.c_int, C.POINTER(C.c_int)]),
        "sim_cavity_stats": (C.c_int, [vp, dp, dp]),
        "sim_redo_count": (C.c_int, [vp, C.POINTER(C.c_longlong)]),
        "sim_set_variant": (C.c_int, [vp, C.c_int, C.c_int]),
        "sim_set_launch_mode": (C.c_int, [vp, C.c_int, C.c_int]),
        "sim_sweep_geometry": (C.c_int, [vp, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_longlong)]),
        "sim_launch_count": (C.c_longlong, [vp]),
        "sim_device_layout": (C.c_int, [vp, C.POINTER(vp), C.POINTER(C.c_longlong), C.POINTER(C.c_int),
                                        C.POINTER(C.c_int), C.POINTER(C.c_int)]),
        "sim_probe_fp64": (C.c_int, [vp, dp, dp]),
        "sim_probe_issue": (C.c_int, [vp, dp]),
        "sim_profiles": (C.c_int, [vp, C.c_double, dp, dp, dp, dp]),
        "sim_qdot_pdf": (C.c_int, [vp, C.c_double, C.c_double, C.c_int, dp, C.POINTER(C.c_longlong)]),
        "sim_qdot_pdf_noalloc": (C.c_int, [vp, C.c_double, C.c_double, C.c_int, dp, C.POINTER(C.c_longlong)]),
        "sim_shock_kinematics": (C.c_int, [vp, dp, dp, C.c_int, C.c_double, dp, dp]),
        "sim_probe_math": (C.c_int, [vp, C.c_int, dp, C.c_int, C.c_double, C.c_double, dp, dp]),
        "sim_profile": (C.c_int, [vp, C.c_int]),
        "sim_kernel_time": (C.c_int, [vp, C.c_int, dp, C.POINTER(C.c_longlong)]),
        "sim_init_slab": (C.c_int, [vp, C.POINTER(Init), C.c_int]),
        "sim_slab_halo_bytes": (C.c_size_t, [vp]),
        "sim_slab_begin": (C.c_int, [vp, C.c_double]),
        "sim_slab_smax_ptr": (C.c_int, [vp, C.POINTER(vp)]),
        "sim_slab_ctl": (C.c_int, [vp, C.c_int]),
        "sim_slab_pass_dir": (C.c_int, [vp, C.c_int]),
        "sim_slab_pass": (C.c_int, [vp, C.c_int]),
        "sim_slab_pack": (C.c_int, [vp, C.c_int, C.c_int, vp]),
        "sim_slab_unpack": (C.c_int, [vp, C.c_int, C.c_int, vp]),
        "sim_slab_info": (C.c_int, [vp, C.POINTER(SlabPeer)]),
        "sim_slab_connect": (C.c_int, [vp, C.c_int, C.POINTER(SlabPeer)]),
        "sim_slab_push": (C.c_int, [vp, C.c_int]),
        "sim_slab_ipc_export": (C.c_int, [vp, vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]),
        "sim_slab_ipc_open": (C.c_int, [vp, C.POINTER(vp)]),
        "sim_slab_ipc_close": (C.c_int, [vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def _fill(struct, d):
    for k, v in d.items():
        setattr(struct, k, v)
    return struct


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def workspace_bytes(grid):
    """sim_workspace_bytes for a grid dict"""
    return int(load_library().sim_workspace_bytes(C.byref(_fill(Grid(), grid))))


class Sim:
    """One simulation on the current CUDA device. grid/eos/kin/init are plain dicts (see `inputs`)."""

    def __init__(self, grid, eos, kin, device=None, variant=None, use_graph=True, library_workspace=False, workspace=None):
        import torch
        self.L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1905_05727_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device if device is not None else "cuda:%d" % torch.cuda.current_device())
        self.grid = _fill(Grid(), grid)
        self.eos = _fill(Eos(), eos)
        self.kin = _fill(Kin(), kin)
        self.nx, self.ny = self.grid.nx, self.grid.ny
        nbytes = int(self.L.sim_workspace_bytes(C.byref(self.grid)))
        if nbytes == 0:
            raise NmsdtError("sim_workspace_bytes", SIM_ERR_ARG, "bad grid")
        self.h = C.c_void_p()
        with torch.cuda.device(self.device):
            # device memory: torch's, unless the workspace must be a cudaMalloc allocation of its own (CUDA IPC export)
            # (workspace: a caller's own 256-byte aligned uint8 tensor of at least sim_workspace_bytes -- e.g. one with guard bands)
            if workspace is not None:
                if workspace.dtype != torch.uint8 or workspace.numel() < nbytes or not workspace.is_contiguous():
                    raise ValueError("workspace must be a contiguous uint8 CUDA tensor of at least %d bytes" % nbytes)
                self.workspace = workspace
            else:
                self.workspace = None if library_workspace else torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device)
            rc = self.L.sim_create(C.byref(self.grid), C.byref(self.eos), C.byref(self.kin),
                                   C.c_void_p(self.workspace.data_ptr() if self.workspace is not None else None),
                                   nbytes if self.workspace is not None else 0, C.c_void_p(self.stream.cuda_stream),
                                   C.byref(self.h))
        if rc != 0:
            raise NmsdtError("sim_create", rc, (self.L.sim_last_error(None) or b"").decode())
        if variant is not None:
            self.set_variant(variant, use_graph)

    # -- plumbing ------------------------------------------------------------------------------------
    def _chk(self, rc, what):
        if rc != 0:
            raise NmsdtError(what, rc, (self.L.sim_last_error(self.h) or b"").decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.sim_destroy(self.h)
            self.h = C.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the calls of include/nmsdt.h ------------------------------------------------------------------
    def init(self, init, x_origin=None):
        """sim_init, or sim_init_slab when x_origin (global column of this slab's first column) is given"""
        d = dict(init)
        cav = d.pop("cavities", None)
        ini = _fill(Init(), d)
        keep = None
        if cav is not None and len(cav) > 0:
            keep = (Cavity * len(cav))(*[Cavity(float(c[0]), float(c[1]), float(c[2])) for c in cav])
            ini.cav = C.cast(keep, C.POINTER(Cavity))
            ini.ncav = len(cav)
        if x_origin is None:
            self._chk(self.L.sim_init(self.h, C.byref(ini)), "sim_init")
        else:
            self._chk(self.L.sim_init_slab(self.h, C.byref(ini), int(x_origin)), "sim_init_slab")

    def init_fields(self, q):
        q = [np.ascontiguousarray(a, dtype=np.float64).reshape(self.ny, self.nx) for a in q]
        ptrs = (C.POINTER(C.c_double) * 7)(*[_dp(a) for a in q])
        self._chk(self.L.sim_init_fields(self.h, ptrs), "sim_init_fields")

    def cfl_dt(self):
        dt = C.c_double()
        self._chk(self.L.sim_cfl_dt(self.h, C.byref(dt)), "sim_cfl_dt")
        return dt.value

    def step(self, n=1):
        self._chk(self.L.sim_step(self.h, int(n)), "sim_step")

    def step_dt(self, n, dt):
        self._chk(self.L.sim_step_dt(self.h, int(n), float(dt)), "sim_step_dt")

    def halo(self, d):
        self._chk(self.L.sim_halo(self.h, int(d)), "sim_halo")

    def sweep(self, d, dt):
        self._chk(self.L.sim_sweep(self.h, int(d), float(dt)), "sim_sweep")

    def source(self, tau):
        self._chk(self.L.sim_source(self.h, float(tau)), "sim_source")

    def diagnostics(self, allow_bad=False):
        d = Diag()
        rc = self.L.sim_diagnostics(self.h, C.byref(d))
        if not (allow_bad and rc == SIM_ERR_BAD):
            self._chk(rc, "sim_diagnostics")
        return {n: getattr(d, n) for n, _ in Diag._fields_}

    def read_field(self, fid):
        if isinstance(fid, str):
            fid = FIELD[fid]
        out = np.empty((self.ny, self.nx), dtype=np.float64)
        self._chk(self.L.sim_read_field(self.h, int(fid), _dp(out)), "sim_read_field")
        return out

    def state(self):
        return [self.read_field(k) for k in range(7)]

    def cavities(self):
        n = C.c_int()
        self._chk(self.L.sim_get_cavities(self.h, None, 0, C.byref(n)), "sim_get_cavities")
        arr = (Cavity * max(n.value, 1))()
        self._chk(self.L.sim_get_cavities(self.h, arr, n.value, C.byref(n)), "sim_get_cavities")
        return np.array([[arr[i].x, arr[i].y, arr[i].r] for i in range(n.value)], dtype=np.float64).reshape(-1, 3)

    def cavity_stats(self):
        """(air fraction asked of the seeded generator, air fraction placed); (0, 0) for a list or a lattice"""
        a, b = C.c_double(), C.c_double()
        self._chk(self.L.sim_cavity_stats(self.h, C.byref(a), C.byref(b)), "sim_cavity_stats")
        return a.value, b.value

    def redo_count(self):
        n = C.c_longlong()
        self._chk(self.L.sim_redo_count(self.h, C.byref(n)), "sim_redo_count")
        return n.value

    def set_variant(self, variant, use_graph=True):
        self._chk(self.L.sim_set_variant(self.h, int(variant), int(bool(use_graph))), "sim_set_variant")

    def set_launch_mode(self, use_graph=True, use_pdl=False):
        self._chk(self.L.sim_set_launch_mode(self.h, int(bool(use_graph)), int(bool(use_pdl))), "sim_set_launch_mode")

    def sweep_geometry(self, d):
        """(segment length, ramp-up cells, blocks per launch) of the fused sweep in direction d"""
        seg, ramp, nb = C.c_int(), C.c_int(), C.c_longlong()
        self._chk(self.L.sim_sweep_geometry(self.h, int(d), C.byref(seg), C.byref(ramp), C.byref(nb)), "sim_sweep_geometry")
        return seg.value, ramp.value, nb.value

    def launch_count(self):
        return int(self.L.sim_launch_count(self.h))

    def probe_fp64(self):
        g, ms = C.c_double(), C.c_double()
        self._chk(self.L.sim_probe_fp64(self.h, C.byref(g), C.byref(ms)), "sim_probe_fp64")
        return g.value, ms.value

    def probe_issue(self):
        """times [ms] of the DFMA + M other instructions probe for M = 0, 4, 8, 16 per 8 DFMA"""
        ms = (C.c_double * 4)()
        self._chk(self.L.sim_probe_issue(self.h, ms), "sim_probe_issue")
        return [ms[i] for i in range(4)]

    def profiles(self, p_front):
        """Eq. 9-11 and the Appendix C front position: (pbar[nx], rhobar[nx], ubar[nx], x_s)"""
        dp = C.POINTER(C.c_double)
        pb, rb, ub = (np.empty(self.nx, dtype=np.float64) for _ in range(3))
        xs = C.c_double()
        self._chk(self.L.sim_profiles(self.h, float(p_front), pb.ctypes.data_as(dp), rb.ctypes.data_as(dp),
                                      ub.ctypes.data_as(dp), C.byref(xs)), "sim_profiles")
        return pb, rb, ub, xs.value

    def qdot_pdf(self, n_lo=2.0, dn=0.02, nbins=400):
        """Eq. 14-16: (mass[nbins], count[nbins])"""
        m = np.empty(nbins, dtype=np.float64)
        c = np.empty(nbins, dtype=np.int64)
        self._chk(self.L.sim_qdot_pdf(self.h, float(n_lo), float(dn), int(nbins), m.ctypes.data_as(C.POINTER(C.c_double)),
                                      c.ctypes.data_as(C.POINTER(C.c_longlong))), "sim_qdot_pdf")
        return m, c

    def qdot_pdf_noalloc(self, n_lo=2.0, dn=0.02, nbins=400):
        """Eq. 14-16 as qdot_pdf, for callers that cannot let the library allocate device memory (the GPU belongs to the
        caller's own arena, or a cudaMalloc's device-wide synchronisation would stall work queued by other handles): the
        scratch is a fixed array inside libnmsdt.so, so nbins <= 512, and calls that may overlap on one GPU must be
        serialised by the caller (include/nmsdt.h: sim_qdot_pdf_noalloc).  Returns (mass[nbins], count[nbins])."""
        m = np.empty(nbins, dtype=np.float64)
        c = np.empty(nbins, dtype=np.int64)
        self._chk(self.L.sim_qdot_pdf_noalloc(self.h, float(n_lo), float(dn), int(nbins), m.ctypes.data_as(C.POINTER(C.c_double)),
                                              c.ctypes.data_as(C.POINTER(C.c_longlong))), "sim_qdot_pdf_noalloc")
        return m, c

    def shock_kinematics(self, t, xs, dtau):
        """Eq. C1-C2: (u_s[n], a_s[n])"""
        dp = C.POINTER(C.c_double)
        t = np.ascontiguousarray(t, dtype=np.float64)
        xs = np.ascontiguousarray(xs, dtype=np.float64)
        us, a = np.empty_like(t), np.empty_like(t)
        self._chk(self.L.sim_shock_kinematics(self.h, t.ctypes.data_as(dp), xs.ctypes.data_as(dp), int(t.size), float(dtau),
                                              us.ctypes.data_as(dp), a.ctypes.data_as(dp)), "sim_shock_kinematics")
        return us, a

    def probe_math(self, fn, x, a=0.0, b=0.0):
        """device evaluation of the fused path's elementary functions (include/nmsdt.h: sim_probe_math)"""
        x = np.ascontiguousarray(x, dtype=np.float64)
        y0, y1 = np.empty_like(x), np.empty_like(x)
        dp = C.POINTER(C.c_double)
        self._chk(self.L.sim_probe_math(self.h, int(fn), x.ctypes.data_as(dp), int(x.size), float(a), float(b),
                                        y0.ctypes.data_as(dp), y1.ctypes.data_as(dp)), "sim_probe_math")
        return y0, y1

    def profile(self, on):
        self._chk(self.L.sim_profile(self.h, int(bool(on))), "sim_profile")

    def kernel_times(self):
        """{kind: (total ms, launches)} accumulated between profile(True) and profile(False)"""
        out = {}
        for name, kid in KERNEL_KINDS.items():
            ms, n = C.c_double(), C.c_longlong()
            self._chk(self.L.sim_kernel_time(self.h, kid, C.byref(ms), C.byref(n)), "sim_kernel_time")
            out[name] = (ms.value, int(n.value))
        return out

    def init_fields_ptr(self, arrays):
        """arrays: 7 C-contiguous float64 numpy arrays (e.g. views of pinned torch tensors); no copy is made"""
        ptrs = (C.POINTER(C.c_double) * 7)(*[_dp(a) for a in arrays])
        self._chk(self.L.sim_init_fields(self.h, ptrs), "sim_init_fields")

    def read_field_into(self, fid, out):
        self._chk(self.L.sim_read_field(self.h, int(fid), _dp(out)), "sim_read_field")

    def synchronize(self):
        self.stream.synchronize()

    # -- slab decomposition (include/nmsdt.h sim_slab_*) ---------------------------------------------------
    def slab_halo_bytes(self):
        return int(self.L.sim_slab_halo_bytes(self.h))

    def slab_begin(self, dt_fixed=0.0):
        self._chk(self.L.sim_slab_begin(self.h, float(dt_fixed)), "sim_slab_begin")

    def slab_smax_ptr(self):
        p = C.c_void_p()
        self._chk(self.L.sim_slab_smax_ptr(self.h, C.byref(p)), "sim_slab_smax_ptr")
        return int(p.value)

    def slab_ctl(self, advance):
        self._chk(self.L.sim_slab_ctl(self.h, int(bool(advance))), "sim_slab_ctl")

    def slab_pass_dir(self, p):
        d = self.L.sim_slab_pass_dir(self.h, int(p))
        if d < 0:
            raise NmsdtError("sim_slab_pass_dir", d, "bad argument")
        return d

    def slab_pass(self, p):
        self._chk(self.L.sim_slab_pass(self.h, int(p)), "sim_slab_pass")

    def slab_pack(self, p, side, dev_ptr):
        self._chk(self.L.sim_slab_pack(self.h, int(p), int(side), C.c_void_p(dev_ptr)), "sim_slab_pack")

    def slab_unpack(self, p, side, dev_ptr):
        self._chk(self.L.sim_slab_unpack(self.h, int(p), int(side), C.c_void_p(dev_ptr)), "sim_slab_unpack")

    def slab_info(self):
        info = SlabPeer()
        self._chk(self.L.sim_slab_info(self.h, C.byref(info)), "sim_slab_info")
        return info

    def slab_connect(self, side, peer):
        self._chk(self.L.sim_slab_connect(self.h, int(side), C.byref(peer) if peer is not None else None), "sim_slab_connect")

    def slab_push(self, p):
        self._chk(self.L.sim_slab_push(self.h, int(p)), "sim_slab_push")

    def slab_ipc_export(self):
        """(64-byte handle, offset of plane set A, offset of plane set B) of a library-allocated workspace"""
        buf = C.create_string_buffer(64)
        oa, ob = C.c_size_t(), C.c_size_t()
        self._chk(self.L.sim_slab_ipc_export(self.h, buf, C.byref(oa), C.byref(ob)), "sim_slab_ipc_export")
        return bytes(buf.raw), int(oa.value), int(ob.value)
