"""Multi-GPU x-slab decomposition of the step (the paper names multi-GPU runs as future
work).  Host-side plumbing only: every arithmetic step runs in the kernels of libnmsdt.so (sim_slab_* calls of
include/nmsdt.h); PyTorch supplies device buffers, streams and `torch.distributed`.

The domain is cut into slabs of whole columns along x (the long axis), one slab per GPU / process.  Per step the
slabs exchange exactly one thing -- the two edge columns of the 7 planes per side before the x-sweep (stencil radius 2;
7 x ny x 2 doubles = 0.46 MB at ny = 4096) -- and agree on the time step through one max-allreduce of the 8-byte
wavespeed word.  The y-sweep and the source step need no communication.  Every slab then computes bit for bit what the
single-GPU run computes for its columns.

Two transports for the halo columns:
  "staged": sim_slab_pack -> isend / irecv (NCCL over NVLink; gloo in the CPU tests) -> sim_slab_unpack
  "peer"  : sim_slab_push writes the edge columns straight into the neighbour's ghost columns through peer memory
            (the neighbour's workspace mapped with CUDA IPC); a one-word allreduce orders push -> sweep.

`DistSlab` is the one-process-per-GPU driver; `LocalSlabs` runs K slabs of one domain one after the other on a single
GPU in one process (no rank ever waits for another: the pushes of all slabs are enqueued before any sweep) -- it is how
the decomposition is checked against the undivided run where only one GPU exists.
"""
import ctypes as C

import numpy as np

BC_PERIODIC, BC_EXTERNAL = 1, 4
NG = 2           # ghost / halo columns per side


# ---- pure host logic (no device, no library) ---------------------------------------------------------------------
def partition(nx, world):
    """[(x_origin, nx_local)] for ranks 0..world-1: contiguous column ranges, sizes differ by at most one."""
    if world < 1 or nx < NG * world:
        raise ValueError("cannot cut %d columns into %d slabs of at least %d columns" % (nx, world, NG))
    base, rem = divmod(nx, world)
    out, x0 = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((x0, n))
        x0 += n
    return out


def neighbours(rank, world, periodic_x):
    """(rank of the x-lo neighbour or None, rank of the x-hi neighbour or None)"""
    if world == 1:
        return None, None
    lo = rank - 1 if rank > 0 else (world - 1 if periodic_x else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic_x else None)
    return lo, hi


def slab_grid(grid, rank, world):
    """(grid dict of this rank's slab, x_origin): sides facing another slab become BC_EXTERNAL."""
    x0, n = partition(grid["nx"], world)[rank]
    lo, hi = neighbours(rank, world, grid["bc_xlo"] == BC_PERIODIC)
    g = dict(grid)
    g["nx"] = n
    if lo is not None:
        g["bc_xlo"] = BC_EXTERNAL
    if hi is not None:
        g["bc_xhi"] = BC_EXTERNAL
    return g, x0


def _as_tensor(ptr, nbytes, dtype, torch, device):
    """zero-copy torch view of `nbytes` at raw pointer `ptr` (device memory of the library, or host memory)"""
    if device.type == "cuda":
        class _Holder:
            pass
        h = _Holder()
        h.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (int(ptr), False), "version": 2}
        return torch.as_tensor(h, device=device).view(dtype)
    arr = np.ctypeslib.as_array(C.cast(C.c_void_p(int(ptr)), C.POINTER(C.c_uint8)), shape=(nbytes,))
    return torch.from_numpy(arr).view(dtype)


def exchange_staged(sim, p, lo, hi, send, recv, dist, group=None, bounce=None):
    """One halo exchange for pass `p`: pack both edges, post all sends / receives at once, unpack the ghosts.
    send / recv: {side: tensor}.  Receives are posted hi first: with two ranks and periodic x both neighbours are the
    same rank, whose first send (its lo edge) is this rank's hi ghost block (NCCL matches point-to-point in order).
    bounce: {("s"|"r", side): CPU tensor} when the backend cannot move device tensors (gloo point-to-point): the blocks
    then travel through host memory."""
    ops = []
    for side, peer in ((0, lo), (1, hi)):
        if peer is not None:
            sim.slab_pack(p, side, send[side].data_ptr())
            buf = send[side]
            if bounce is not None:
                bounce[("s", side)].copy_(send[side])                    # synchronises with the pack kernel
                buf = bounce[("s", side)]
            ops.append(dist.P2POp(dist.isend, buf, peer, group=group, tag=side))
    for side, peer in ((1, hi), (0, lo)):
        if peer is not None:
            buf = recv[side] if bounce is None else bounce[("r", side)]
            ops.append(dist.P2POp(dist.irecv, buf, peer, group=group, tag=1 - side))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    for side, peer in ((0, lo), (1, hi)):
        if peer is not None:
            if bounce is not None:
                recv[side].copy_(bounce[("r", side)])
            sim.slab_unpack(p, side, recv[side].data_ptr())


# ---- one process per GPU ------------------------------------------------------------------------------------------
class DistSlab:
    """This rank's slab of a domain cut over the ranks of a torch.distributed group.

    `sim_factory(grid_dict)` returns the object that implements the sim_slab_* calls for the slab's grid (a
    `binding.Sim`; the CPU tests pass a stand-in with the same methods), already created on `device`."""

    def __init__(self, grid, sim_factory, dist, device, transport="staged", group=None):
        import torch
        self.torch, self.dist, self.group = torch, dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.global_grid = dict(grid)
        self.grid, self.x0 = slab_grid(grid, self.rank, self.world)
        self.lo, self.hi = neighbours(self.rank, self.world, grid["bc_xlo"] == BC_PERIODIC)
        self.device = torch.device(device)
        self.sim = sim_factory(self.grid)
        nb = self.sim.slab_halo_bytes()
        mk = lambda: torch.empty(nb // 8, dtype=torch.float64, device=self.device)          # noqa: E731
        self.send = {s: mk() for s, p in ((0, self.lo), (1, self.hi)) if p is not None}
        self.recv = {s: mk() for s, p in ((0, self.lo), (1, self.hi)) if p is not None}
        self.smax = _as_tensor(self.sim.slab_smax_ptr(), 8, torch.int64, torch, self.device)
        self.token = torch.zeros(1, dtype=torch.int64, device=self.device)                 # barrier word of the peer transport
        self.transport = transport
        self.bounce = None
        if self.device.type == "cuda" and dist.get_backend(group) == "gloo":     # gloo point-to-point moves host memory only
            self.bounce = {(k, s): torch.empty(nb // 8, dtype=torch.float64).pin_memory() for k in "sr" for s in self.send}
        self._ipc_open = []
        if transport == "peer" and self.world > 1:
            self._connect_peers()
        elif transport not in ("staged", "peer"):
            raise ValueError("transport must be 'staged' or 'peer'")
        self._begun = None

    def _connect_peers(self):
        """exchange CUDA IPC handles of the workspaces and map the neighbours' plane sets into this process"""
        from .binding import SlabPeer, load_library
        L = load_library()
        info = self.sim.slab_info()
        handle, off_a, off_b = self.sim.slab_ipc_export()
        mine = dict(handle=handle, off=(off_a, off_b), stride=int(info.plane_stride), pitch=int(info.pitch), nx=int(info.nx),
                    ny=int(info.ny))
        everyone = [None] * self.world
        self.dist.all_gather_object(everyone, mine, group=self.group)
        opened = {}
        for side, peer in ((0, self.lo), (1, self.hi)):
            if peer is None:
                continue
            d = everyone[peer]
            if peer not in opened:
                base = C.c_void_p()
                rc = L.sim_slab_ipc_open(C.create_string_buffer(d["handle"], 64), C.byref(base))
                if rc != 0:
                    raise RuntimeError("sim_slab_ipc_open failed (%d): %s" % (rc, (L.sim_last_error(None) or b"").decode()))
                opened[peer] = int(base.value)
                self._ipc_open.append(int(base.value))
            p = SlabPeer()
            p.plane0[0], p.plane0[1] = opened[peer] + d["off"][0], opened[peer] + d["off"][1]
            p.plane_stride, p.pitch, p.nx, p.ny = d["stride"], d["pitch"], d["nx"], d["ny"]
            self.sim.slab_connect(side, p)

    def init(self, init):
        """problem setup of the WHOLE domain (global cell units); every rank paints its own columns"""
        self.sim.init(init, x_origin=self.x0)
        self._begun = None

    def _allreduce_smax(self):
        if self.world > 1:
            self.dist.all_reduce(self.smax, op=self.dist.ReduceOp.MAX, group=self.group)

    def _exchange(self, p):
        if self.world == 1:
            return
        if self.transport == "staged":
            exchange_staged(self.sim, p, self.lo, self.hi, self.send, self.recv, self.dist, self.group, self.bounce)
        else:
            # every rank stores its edge columns into its neighbours' ghost columns, then all ranks meet: when the
            # allreduce has finished on this stream, the neighbours' push kernels (enqueued before theirs) are complete.
            # The ghost columns written here were last read one step ago, before the end-of-step allreduce.
            self.sim.slab_push(p)
            self.dist.all_reduce(self.token, group=self.group)

    def step(self, n=1, dt_fixed=0.0):
        """n steps (CFL-limited, or with the fixed dt); asynchronous like sim_step"""
        if self._begun != dt_fixed:
            self.sim.slab_begin(dt_fixed)
            self._allreduce_smax()
            self.sim.slab_ctl(0)
            self._begun = dt_fixed
        for _ in range(n):
            for p in (1, 2):
                if self.sim.slab_pass_dir(p) == 0:
                    self._exchange(p)
                self.sim.slab_pass(p)
            self._allreduce_smax()
            self.sim.slab_ctl(1)

    def diagnostics(self):
        """global diagnostics: integrals summed, S_max / bad flag maximised over the slabs (same dict as Sim.diagnostics)"""
        d = self.sim.diagnostics(allow_bad=True)
        keys = ["M2r", "M2tot0", "burned_mass", "rate_inst", "mass1", "mass2", "momx", "momy", "energy"]
        if self.world > 1:
            t = self.torch.tensor([d[k] for k in keys], dtype=self.torch.float64, device=self.device)
            m = self.torch.tensor([d["smax"], float(d["bad_state"])], dtype=self.torch.float64, device=self.device)
            self.dist.all_reduce(t, group=self.group)
            self.dist.all_reduce(m, op=self.dist.ReduceOp.MAX, group=self.group)
            for k, v in zip(keys, t.tolist()):
                d[k] = v
            d["smax"], d["bad_state"] = m[0].item(), int(m[1].item())
        return d

    def close(self):
        from .binding import load_library
        for side in (0, 1):
            if self.transport == "peer" and self.world > 1:
                self.sim.slab_connect(side, None)
        self.sim.synchronize()
        for base in self._ipc_open:
            load_library().sim_slab_ipc_close(C.c_void_p(base))
        self._ipc_open = []
        self.sim.close()


# ---- K slabs of one domain in one process on one GPU ---------------------------------------------------------------
class LocalSlabs:
    """The decomposed step with all K slabs on the current GPU, driven in stream order by one process: every slab's
    exchange kernels are enqueued before any slab's sweep, so no kernel waits for another.  Used to check the decomposition
    (same halo kernels, same step pieces as DistSlab) against the undivided run on a single GPU."""

    def __init__(self, grid, eos, kin, k, transport="peer", device=None):
        import torch
        from .binding import Sim
        self.torch, self.k, self.transport = torch, k, transport
        self.parts = partition(grid["nx"], k)
        per = grid["bc_xlo"] == BC_PERIODIC
        self.nb = [neighbours(r, k, per) for r in range(k)]
        self.sims = [Sim(slab_grid(grid, r, k)[0], eos, kin, device=device) for r in range(k)]
        self.device = self.sims[0].device
        self.smax = [_as_tensor(s.slab_smax_ptr(), 8, torch.int64, torch, self.device) for s in self.sims]
        if transport == "peer":
            infos = [s.slab_info() for s in self.sims]
            for r, s in enumerate(self.sims):
                for side in (0, 1):
                    if self.nb[r][side] is not None:
                        s.slab_connect(side, infos[self.nb[r][side]])
        else:
            n = self.sims[0].slab_halo_bytes() // 8
            self.buf = {(r, side): torch.empty(n, dtype=torch.float64, device=self.device)
                        for r in range(k) for side in (0, 1) if self.nb[r][side] is not None}
        self._begun = None

    def init(self, init):
        for s, (x0, _) in zip(self.sims, self.parts):
            s.init(init, x_origin=x0)
        self._begun = None

    def _max_smax(self):
        m = self.torch.stack(self.smax).max()
        for t in self.smax:
            t.fill_(m)

    def _exchange(self, p):
        if self.transport == "peer":
            for s in self.sims:
                s.slab_push(p)
            return
        for r, s in enumerate(self.sims):
            for side in (0, 1):
                if self.nb[r][side] is not None:
                    s.slab_pack(p, side, self.buf[(r, side)].data_ptr())
        for r, s in enumerate(self.sims):
            for side in (0, 1):
                if self.nb[r][side] is not None:          # my side-ghosts = the neighbour's opposite edge
                    s.slab_unpack(p, side, self.buf[(self.nb[r][side], 1 - side)].data_ptr())

    def step(self, n=1, dt_fixed=0.0):
        if self._begun != dt_fixed:
            for s in self.sims:
                s.slab_begin(dt_fixed)
            self._max_smax()
            for s in self.sims:
                s.slab_ctl(0)
            self._begun = dt_fixed
        for _ in range(n):
            for p in (1, 2):
                if self.sims[0].slab_pass_dir(p) == 0:
                    self._exchange(p)
                for s in self.sims:
                    s.slab_pass(p)
            self._max_smax()
            for s in self.sims:
                s.slab_ctl(1)

    def state(self):
        """the 7 conserved planes of the whole domain, slabs joined along x"""
        per = [s.state() for s in self.sims]
        return [np.concatenate([per[r][f] for r in range(self.k)], axis=1) for f in range(7)]

    def diagnostics(self):
        ds = [s.diagnostics(allow_bad=True) for s in self.sims]
        d = dict(ds[0])
        for key in ("M2r", "M2tot0", "burned_mass", "rate_inst", "mass1", "mass2", "momx", "momy", "energy"):
            d[key] = sum(x[key] for x in ds)
        d["smax"] = max(x["smax"] for x in ds)
        d["bad_state"] = max(x["bad_state"] for x in ds)
        return d

    def close(self):
        for s in self.sims:
            s.close()
