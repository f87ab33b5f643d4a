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

    def _get(self, what):
        s = self.solver
        return (s.halo_get(FACE_ZLO, what) if self.lo is not None else None,
                s.halo_get(FACE_ZHI, what) if self.hi is not None else None)

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

    def _exchange(self, what):
        send_lo, send_hi = self._get(what)
        recv_lo, recv_hi = self._buffers(what)
        self.solver.torch.cuda.current_stream().synchronize()     # the messages are complete before they leave
        self.transport.exchange(send_lo, send_hi, recv_lo, recv_hi)
        self._put(what, recv_lo, recv_hi)

    def set_state(self, rho, u, v, w, p, psi):
        """Arrays of THIS slab, (z1 - z0, ny, nx)."""
        self.solver.set_state(rho, u, v, w, p, psi)
        if self.lo is not None or self.hi is not None:
            self._exchange(cspt.HALO_PSI)
            self.solver.finish_state()

    def step_cfl(self, cfl):
        s = self.solver
        s.fill_ghosts()
        self._exchange(cspt.HALO_U)
        t = s.torch.tensor([s.compute_dt(cfl)], dtype=s.torch.float64, device=s.device)
        dt = float(self.transport.min_scalar(t).item())
        s.step_filled(dt)
        return dt

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

    def step_cfl(self, cfl):
        for sl in self.slabs:
            sl.solver.fill_ghosts()
        self._exchange(cspt.HALO_U)
        dt = min(sl.solver.compute_dt(cfl) for sl in self.slabs)
        for sl in self.slabs:
            sl.solver.step_filled(dt)
        return dt

    def get_conserved(self):
        torch = self.slabs[0].solver.torch
        parts = [sl.solver.get_conserved() for sl in self.slabs]
        return [torch.cat([p[f] for p in parts], dim=0) for f in range(5)]

    def close(self):
        for sl in self.slabs:
            sl.solver.close()
