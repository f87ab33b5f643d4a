"""Host side of the z-slab decomposition (paper_1912_04855_b200/slab.py): the partition, the
neighbour table, the boundary kinds of a slab, and the torch.distributed transport with two and three gloo ranks on
the CPU (the message order that two ranks on a periodic axis rely on, and the min-reduction of the time step)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1912_04855_b200 import cspt, slab

P, O, I, X = cspt.BC_PERIODIC, cspt.BC_OUTFLOW, cspt.BC_INFLOW, cspt.BC_EXTERNAL


def test_partition_covers_the_axis_evenly():
    assert slab.partition(26, 3) == [(0, 9), (9, 18), (18, 26)]
    assert slab.partition(512, 4) == [(0, 128), (128, 256), (256, 384), (384, 512)]
    assert slab.partition(8, 1) == [(0, 8)]
    for nz, world in ((1024, 8), (100, 7), (33, 8)):
        parts = slab.partition(nz, world)
        assert parts[0][0] == 0 and parts[-1][1] == nz
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 4
    with pytest.raises(ValueError):
        slab.partition(15, 4)          # a slab must hold the 3-plane halo it sends and 4 planes for a non-periodic ctx


def test_neighbours_and_slab_bc():
    per, out = (P,) * 6, (I, O, P, P, O, I)
    assert slab.neighbours(per, 0, 4) == (3, 1) and slab.neighbours(per, 3, 4) == (2, 0)
    assert slab.neighbours(per, 0, 1) == (0, 0)                         # one periodic slab wraps onto itself
    assert slab.neighbours(out, 0, 4) == (None, 1) and slab.neighbours(out, 3, 4) == (2, None)
    assert slab.neighbours(out, 0, 1) == (None, None)
    assert slab.slab_bc(per, 1, 4) == [P, P, P, P, X, X]
    assert slab.slab_bc(out, 0, 4) == [I, O, P, P, O, X]                # the physical face keeps the grid's kind
    assert slab.slab_bc(out, 3, 4) == [I, O, P, P, X, I]
    assert slab.slab_bc(out, 0, 1) == list(out)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, bc, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    tr = slab.DistTransport(bc, rank, world)
    n = 7
    send_lo = torch.full((n,), 10.0 * rank + 1.0, dtype=torch.float64)       # "my lo planes"
    send_hi = torch.full((n,), 10.0 * rank + 2.0, dtype=torch.float64)       # "my hi planes"
    recv_lo = torch.zeros(n, dtype=torch.float64) if tr.lo is not None else None
    recv_hi = torch.zeros(n, dtype=torch.float64) if tr.hi is not None else None
    tr.exchange(send_lo if tr.lo is not None else None, send_hi if tr.hi is not None else None, recv_lo, recv_hi)
    dt = tr.min_scalar(torch.tensor([0.5 - 0.1 * rank], dtype=torch.float64))
    # the signal-speed word of the sync-free protocol: reduced IN PLACE on a view of a larger buffer, in both dtypes
    ws = torch.zeros(16, dtype=torch.uint8)
    word = ws[8:16].view(torch.float64)
    word[0] = 1.0 + 0.25 * rank
    tr.max_scalar(word)
    w32 = ws[0:4].view(torch.float32)
    w32[0] = 3.0 - rank
    tr.max_scalar(w32)
    assert not tr.stream_ordered                     # gloo: SlabSolver synchronises before it hands messages over
    out[rank] = (None if recv_lo is None else float(recv_lo[0]), None if recv_hi is None else float(recv_hi[0]),
                 float(dt[0]), float(ws[8:16].view(torch.float64)[0]), float(ws[0:4].view(torch.float32)[0]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True)])
def test_transport_delivers_the_right_planes(world, periodic):
    bc = (P,) * 6 if periodic else (P, P, P, P, O, O)
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), bc, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        lo, hi = slab.neighbours(bc, r, world)
        got_lo, got_hi, dt, smax64, smax32 = res[r]
        assert smax64 == 1.0 + 0.25 * (world - 1) and smax32 == 3.0      # maxima over the ranks, in place
        # my lo ghost planes are the HI planes of the rank below, my hi ghost planes the LO planes of the rank above
        assert got_lo == (None if lo is None else 10.0 * lo + 2.0)
        assert got_hi == (None if hi is None else 10.0 * hi + 1.0)
        assert dt == pytest.approx(0.5 - 0.1 * (world - 1))


def test_single_periodic_slab_wraps_without_a_process_group():
    tr = slab.DistTransport((P,) * 6, 0, 1)
    a, b = torch.ones(3), 2 * torch.ones(3)
    rl, rh = torch.zeros(3), torch.zeros(3)
    tr.exchange(a, b, rl, rh)
    assert torch.equal(rl, b) and torch.equal(rh, a)
    assert float(tr.min_scalar(torch.tensor([0.25]))[0]) == 0.25
    assert float(tr.max_scalar(torch.tensor([0.25]))[0]) == 0.25 and not tr.stream_ordered
