"""CPU stand-in for the sim_slab_* calls of include/nmsdt.h, used only by the world_size-2 gloo tests of
paper_1905_05727_b200/slab.py (the real calls need a GPU).  It has the same protocol -- ping-pong plane sets A / B,
pass direction alternating with the step parity, radius-2 stencil in x that reads two ghost columns per side, an
ordered-bits max word, a control step that turns the (all-reduced) max into the next dt -- but a made-up, cheap,
nonlinear update, so that a wrong neighbour, a swapped side, a stale ghost column or a missing max-reduction changes the
result.  None of the paper's arithmetic is here."""
import ctypes as C

import numpy as np

NG, NF = 2, 7


class StandInSim:
    def __init__(self, grid, x_origin_hint=None):
        self.nx, self.ny = grid["nx"], grid["ny"]
        self.bc = (grid["bc_xlo"], grid["bc_xhi"])
        self.cfl = grid["cfl"]
        self.A = np.zeros((NF, self.ny, self.nx + 2 * NG))
        self.B = np.zeros_like(self.A)
        self.word = np.zeros(1, dtype=np.int64)
        self.dt, self.dt_fixed, self.t, self.step_no = 0.0, 0.0, 0.0, 0
        self.device = None

    # -- setup: a smooth global field sampled on this slab's columns -------------------------------------------------
    def init(self, init, x_origin=0):
        i = np.arange(self.nx) + x_origin
        j = np.arange(self.ny)[:, None]
        for f in range(NF):
            self.A[f, :, NG:-NG] = 1.0 + 0.3 * np.sin(0.37 * i + 0.11 * f) * np.cos(0.23 * j) + 0.01 * f + init.get("bump", 0.0) * (i == 5)
        self.t, self.step_no = 0.0, 0

    # -- the protocol ------------------------------------------------------------------------------------------------
    def slab_halo_bytes(self):
        return NF * self.ny * NG * 8

    def slab_smax_ptr(self):
        return self.word.ctypes.data

    def _local_max(self, u):
        self.word[0] = np.abs(u[:, :, NG:-NG]).max().view(np.int64)

    def slab_begin(self, dt_fixed):
        self.dt_fixed = dt_fixed
        self._local_max(self.A)

    def slab_ctl(self, advance):
        if advance:
            self.t += self.dt
            self.step_no += 1
        smax = self.word.view(np.float64)[0]
        self.dt = self.dt_fixed if self.dt_fixed > 0 else self.cfl / smax
        self.word[0] = 0

    def slab_pass_dir(self, p):
        d1 = self.step_no & 1
        return d1 if p == 1 else 1 - d1

    def _fill_local_ghosts(self, u):
        for side, bc in enumerate(self.bc):
            if bc == 4:                 # external: the neighbour's columns, already in place
                continue
            for m in range(NG):
                if side == 0:
                    u[:, :, NG - 1 - m] = u[:, :, -NG - 1 - m] if bc == 1 else u[:, :, NG]
                else:
                    u[:, :, -NG + m] = u[:, :, NG + m] if bc == 1 else u[:, :, -NG - 1]

    def slab_pass(self, p):
        src, dst = (self.A, self.B) if p == 1 else (self.B, self.A)
        if self.slab_pass_dir(p) == 0:
            self._fill_local_ghosts(src)
            c = src[:, :, NG:-NG]
            lap = src[:, :, :-4] - 4 * src[:, :, 1:-3] + 6 * c - 4 * src[:, :, 3:-1] + src[:, :, 4:]
            dst[:, :, NG:-NG] = c - self.dt * (0.05 * lap + 0.2 * c * (src[:, :, 3:-1] - src[:, :, 1:-3]))
        else:
            c = src[:, :, NG:-NG]
            dst[:, :, NG:-NG] = c + self.dt * 0.1 * (np.roll(c, 1, axis=1) - 2 * c + np.roll(c, -1, axis=1))
        if p == 2:
            self._local_max(dst)

    def _block(self, ptr):
        return np.ctypeslib.as_array(C.cast(C.c_void_p(int(ptr)), C.POINTER(C.c_double)), shape=(NF, self.ny, NG))

    def slab_pack(self, p, side, ptr):
        u = self.A if p == 1 else self.B
        self._block(ptr)[...] = u[:, :, NG:2 * NG] if side == 0 else u[:, :, -2 * NG:-NG]

    def slab_unpack(self, p, side, ptr):
        u = self.A if p == 1 else self.B
        if side == 0:
            u[:, :, :NG] = self._block(ptr)
        else:
            u[:, :, -NG:] = self._block(ptr)

    def diagnostics(self, allow_bad=False):
        s = float(self.A[:, :, NG:-NG].sum())
        d = dict(t=self.t, step=self.step_no, dt_last=self.dt, smax=float(np.abs(self.A[:, :, NG:-NG]).max()), bad_state=0)
        for k in ("M2r", "M2tot0", "burned_mass", "rate_inst", "mass1", "mass2", "momx", "momy", "energy"):
            d[k] = s
        return d

    def state(self):
        return self.A[:, :, NG:-NG].copy()

    def synchronize(self):
        pass

    def close(self):
        pass
