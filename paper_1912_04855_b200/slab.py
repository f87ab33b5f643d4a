"""z-slab decomposition of one grid over several GPUs, one process per GPU (
PAPER.md:106 "the computational domain is divided between GPUs", :123).

Host-side plumbing only: every step of the method runs in the kernels of libcspt.so.  A slab is a cspt.Solver whose z
faces towards other slabs have kind BC_EXTERNAL; per step the three ghost planes of the five conserved fields cross
each such face once (NCCL send/recv over NVLink through torch.distributed) and one scalar min-reduction fixes the
time step, after which the slabs advance exactly as the undivided grid does (include/cspt.h, "z-slab decomposition").

    SlabSolver   one rank's slab + a torch.distributed transport       (the multi-GPU path)
    LocalSlabs   all slabs of a grid in ONE process on one GPU, halos handed over as tensors: the same phases in
                 the same order, used to check the decomposition against the undivided solver where only one GPU
                 is to be had
"""
from . import cspt

FACE_ZLO, FACE_ZHI = 4, 5


# ---- pure host logic (covered by the CPU tests) -----------------------------------------------------------------
def partition(nz, world):
    """[z0, z1) of every rank: as even as possible, lower ranks take the remainder; every slab needs >= 4 planes."""
    if world < 1 or nz < 4 * world:
        raise ValueError("need at least 4 planes per slab: nz=%d world=%d" % (nz, world))
    base, rem = divmod(nz, world)
    out, z = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((z, z + n))
        z += n
    return out


def neighbours(bc, rank, world):
    """(rank below, rank above) across the z faces of this slab, None where the face is a physical boundary."""
    periodic = bc[4] == cspt.BC_PERIODIC
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return lo, hi


def slab_bc(bc, rank, world):
    """Boundary kinds of the slab: a z face with a neighbour becomes BC_EXTERNAL, the others keep the grid's kind."""
    lo, hi = neighbours(bc, rank, world)
    out = list(bc)
    if lo is not None:
        out[4] = cspt.BC_EXTERNAL
    if hi is not None:
        out[5] = cspt.BC_EXTERNAL
    return out


class DistTransport:
    """Halo exchange and min-reduction over torch.distributed (nccl on GPUs, gloo in the CPU tests).

    Every rank posts, in this order, send(lo planes -> rank below), send(hi planes -> rank above),
    recv(hi ghost <- rank above), recv(lo ghost <- rank below): with two ranks on a periodic axis both messages go
    to the same peer and are matched by that order (its first send, the lo planes, is my first receive)."""

    def __init__(self, bc, rank, world, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = rank, world
        self.lo, self.hi = neighbours(bc, rank, world)

    def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
        """send_*: this slab's interior planes next to the face; recv_*: buffers for the ghost planes (None where the
        face has no neighbour).  Returns when the receive buffers are filled."""
        dist = self.dist
        ops = []
        if self.lo == self.rank and self.hi == self.rank:          # one slab, periodic: its own planes wrap around
            recv_hi.copy_(send_lo)
            recv_lo.copy_(send_hi)
            return
        if self.lo is not None:
            ops.append(dist.P2POp(dist.isend, send_lo, self.lo, self.group))
        if self.hi is not None:
            ops.append(dist.P2POp(dist.isend, send_hi, self.hi, self.group))
        if self.hi is not None:
            ops.append(dist.P2POp(dist.irecv, recv_hi, self.hi, self.group))
        if self.lo is not None:
            ops.append(dist.P2POp(dist.irecv, recv_lo, self.lo, self.group))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()

    @property
    def stream_ordered(self):
        """True when the backend enqueues its transfers on CUDA streams ordered after torch's current stream (NCCL)."""
        try:
            return self.world > 1 and self.dist.get_backend(self.group) == "nccl"
        except Exception:
            return False

    def max_scalar(self, t):
        """In-place maximum over all ranks of a one-element tensor."""
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
        return t

    def min_scalar(self, t):
        """In-place minimum over all ranks of a one-element tensor."""
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN, group=self.group)
        return t


# ---- one slab ------------------------------------------------------------------------------------------------------
class _Slab:
    """The phases of one slab; SlabSolver and LocalSlabs only differ in who carries the messages."""

    def __init__(self, nx, ny, nz_global, h, gamma, bc, dtype, rank, world, stream=None):
        self.rank, self.world, self.bc = rank, world, list(bc)
        self.z0, self.z1 = partition(nz_global, world)[rank]
        self.lo, self.hi = neighbours(bc, rank, world)
        self.solver = cspt.Solver(nx, ny, self.z1 - self.z0, h, gamma, slab_bc(bc, rank, world), dtype, stream)

    def local(self, fields):
        """This slab's planes of arrays given on the whole grid (nz, ny, nx)."""
        return [f[self.z0:self.z1] for f in fields]

    def _get(self, what, out=(None, None)):
        s = self.solver
        return (s.halo_get(FACE_ZLO, what, out[0]) if self.lo is not None else None,
                s.halo_get(FACE_ZHI, what, out[1]) if self.hi is not None else None)

    def _put(self, what, recv_lo, recv_hi):
        if self.lo is not None:
            self.solver.halo_put(FACE_ZLO, recv_lo, what)
        if self.hi is not None:
            self.solver.halo_put(FACE_ZHI, recv_hi, what)

    def _buffers(self, what):
        s = self.solver
        mk = lambda: s.torch.empty(s.halo_elems(what), dtype=s.tdtype, device=s.device)
        return (mk() if self.lo is not None else None, mk() if self.hi is not None else None)


class SlabSolver(_Slab):
    """One rank of a z-slab decomposition.  `transport` defaults to torch.distributed's default group."""

    def __init__(self, nx, ny, nz_global, h, gamma, bc, dtype=cspt.F64, rank=0, world=1, transport=None, stream=None):
        super().__init__(nx, ny, nz_global, h, gamma, bc, dtype, rank, world, stream)
        self.transport = transport or DistTransport(bc, rank, world)
        self._bufs = {}

    def _exchange(self, what):
        # message buffers are allocated once per kind of message and reused every step
        if what not in self._bufs:
            self._bufs[what] = (self._buffers(what), self._buffers(what))
        send, recv = self._bufs[what]
        send_lo, send_hi = self._get(what, send)
        # NCCL orders its send/recv after the work already enqueued on torch's current stream (which halo_get made
        # wait for the solver's stream) and makes that stream wait for their completion: no host synchronisation.
        # Any other backend gets the messages only once they are complete.
        if not getattr(self.transport, "stream_ordered", False):
            self.solver.torch.cuda.current_stream().synchronize()
        self.transport.exchange(send_lo, send_hi, recv[0], recv[1])
        self._put(what, recv[0], recv[1])

    def set_state(self, rho, u, v, w, p, psi):
        """Arrays of THIS slab, (z1 - z0, ny, nx)."""
        self.solver.set_state(rho, u, v, w, p, psi)
        if self.lo is not None or self.hi is not None:
            self._exchange(cspt.HALO_PSI)
            self.solver.finish_state()

    def step_cfl(self, cfl, want_dt=True):
        """One CFL-limited step of the whole grid.  The time step never visits the host: the slab's maximum signal
        speed is max-reduced over the ranks in place on the device (a view of the word in the solver's workspace) and
        cspt_step_filled_cfl forms dt from it.  want_dt=False enqueues only (no host synchronisation in the step);
        want_dt=True (default) also returns dt, which waits for the step."""
        s = self.solver
        s.fill_ghosts()
        self._exchange(cspt.HALO_U)
        smax = s.smax_device()
        self.transport.max_scalar(smax)
        s.stream.wait_stream(s.torch.cuda.current_stream())     # the reduced word is in place before dt is formed
        return s.step_filled_cfl(cfl, want_dt)

    def get_conserved(self):
        return self.solver.get_conserved()

    def close(self):
        self.solver.close()


class LocalSlabs:
    """All `world` slabs of a grid in one process on the current GPU (no torch.distributed): the phases of
    SlabSolver.step_cfl run slab after slab and the halo messages are handed over as tensors."""

    def __init__(self, nx, ny, nz_global, h, gamma, bc, dtype=cspt.F64, world=2):
        self.world = world
        self.slabs = [_Slab(nx, ny, nz_global, h, gamma, bc, dtype, r, world) for r in range(world)]

    def _exchange(self, what):
        sent = [sl._get(what) for sl in self.slabs]
        for sl in self.slabs:
            recv_lo = sent[sl.lo][1] if sl.lo is not None else None      # the hi planes of the slab below
            recv_hi = sent[sl.hi][0] if sl.hi is not None else None      # the lo planes of the slab above
            sl._put(what, recv_lo, recv_hi)

    def set_state(self, rho, u, v, w, p, psi):
        """Arrays of the WHOLE grid, (nz, ny, nx)."""
        for sl in self.slabs:
            sl.solver.set_state(*sl.local([rho, u, v, w, p, psi]))
        if self.slabs[0].lo is not None or self.slabs[0].hi is not None:
            self._exchange(cspt.HALO_PSI)
            for sl in self.slabs:
                sl.solver.finish_state()

    def step_cfl(self, cfl, device_dt=False):
        """device_dt=False: dt = min over slabs of cspt_compute_dt on the host, then cspt_step_filled(dt).
        device_dt=True: the phases of SlabSolver.step_cfl: the slabs' signal-speed words are max-reduced on the device
        (here a torch.maximum over the views, standing in for the all-reduce) and cspt_step_filled_cfl forms dt."""
        for sl in self.slabs:
            sl.solver.fill_ghosts()
        self._exchange(cspt.HALO_U)
        if not device_dt:
            dt = min(sl.solver.compute_dt(cfl) for sl in self.slabs)
            for sl in self.slabs:
                sl.solver.step_filled(dt)
            return dt
        words = [sl.solver.smax_device() for sl in self.slabs]
        top = words[0].clone()
        for wd in words[1:]:
            top = self.slabs[0].solver.torch.maximum(top, wd)
        for wd in words:
            wd.copy_(top)
        dts = []
        for sl in self.slabs:
            sl.solver.stream.wait_stream(sl.solver.torch.cuda.current_stream())
            dts.append(sl.solver.step_filled_cfl(cfl, want_dt=True))
        assert all(d == dts[0] for d in dts)
        return dts[0]

    def get_conserved(self):
        torch = self.slabs[0].solver.torch
        parts = [sl.solver.get_conserved() for sl in self.slabs]
        return [torch.cat([p[f] for p in parts], dim=0) for f in range(5)]

    def close(self):
        for sl in self.slabs:
            sl.solver.close()
