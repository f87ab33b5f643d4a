"""z-slab decomposition on ONE GPU: all slabs of a grid live in one
process (paper_1912_04855_b200.slab.LocalSlabs: the phases of the multi-GPU path, messages handed over as tensors,
no kernel waits for another).  The slabs must advance exactly as the undivided solver does (bit for bit: the same
kernels see the same ghost layers), and therefore match the oracle to the tolerance of the undivided path."""
import numpy as np
import pytest

from oracle_util import make_oracle
from paper_1912_04855_b200 import workloads as wl
from test_gpu_parity import field_errors

pytestmark = pytest.mark.gpu
P, O, I = wl.PERIODIC, wl.OUTFLOW, wl.INFLOW


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1912_04855_b200 import build, cspt, slab
    build.build()
    cspt.lib()
    return cspt, slab


def _run_both(cspt, slab, w, world, steps, dtype=None, device_dt=False):
    d = cspt.F64 if (dtype or w.dtype) == "f64" else cspt.F32
    f = w.fields() if dtype is None else [a.astype(np.float32 if dtype == "f32" else np.float64) for a in w.fields()]
    one = cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, d)
    one.set_state(*f)
    many = slab.LocalSlabs(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, d, world)
    many.set_state(*f)
    dts = []
    for _ in range(steps):
        dt1 = one.step_cfl(w.cfl, want_dt=True)
        dt2 = many.step_cfl(w.cfl, device_dt=device_dt)
        assert dt1 == dt2                     # min over the slabs of the local CFL steps is the grid's step, bit for bit
        dts.append(dt1)
    a = [t.cpu().numpy() for t in one.get_conserved()]
    b = [t.cpu().numpy() for t in many.get_conserved()]
    one.close()
    many.close()
    return f, a, b, dts


@pytest.mark.parametrize("world", [1, 2, 3])
@pytest.mark.parametrize("bc", [(P, P, P, P, P, P), (I, O, P, P, O, O), (O, O, O, O, I, O)])
def test_slabs_advance_exactly_as_the_undivided_grid(mods, bc, world):
    cspt, slab = mods
    w = wl.random_smooth(40, 12, 26, bc=bc)          # ragged: 26 planes over 3 slabs = 9 + 9 + 8
    _, a, b, _ = _run_both(cspt, slab, w, world, 10)
    for q in range(5):
        assert np.array_equal(a[q], b[q]), (q, float(np.max(np.abs(a[q] - b[q]))))


@pytest.mark.parametrize("world,bc,dtype", [(2, (P, P, P, P, P, P), None), (3, (I, O, P, P, O, O), None),
                                            (3, (O, O, O, O, I, O), "f32")])
def test_time_step_reduced_on_the_device(mods, world, bc, dtype):
    """The sync-free protocol of SlabSolver.step_cfl (cspt_smax_device -> max over the slabs in place ->
    cspt_step_filled_cfl) gives the time step and the state of the undivided grid, bit for bit."""
    cspt, slab = mods
    w = wl.random_smooth(40, 12, 26, bc=bc)
    _, a, b, _ = _run_both(cspt, slab, w, world, 8, dtype=dtype, device_dt=True)
    for q in range(5):
        assert np.array_equal(a[q], b[q]), q


def _nccl_rank(rank, world, port, nz, out_path):
    import os
    import torch
    import torch.distributed as dist
    from paper_1912_04855_b200 import cspt, slab
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    w = wl.random_smooth(40, 12, nz, bc=(P, P, P, P, P, P))
    s = slab.SlabSolver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, cspt.F64, rank, world)
    s.set_state(*s.local(w.fields()))
    dts = [s.step_cfl(w.cfl) for _ in range(6)]
    s.step_cfl(w.cfl, want_dt=False)                  # the sync-free form
    dts.append(None)
    mine = torch.stack(s.get_conserved()).cpu()
    torch.save({"z0": s.z0, "z1": s.z1, "U": mine, "dts": dts}, "%s.%d" % (out_path, rank))
    s.close()
    dist.destroy_process_group()


def test_slab_solver_over_nccl_on_two_gpus(mods, tmp_path):
    """The real transport: one process per GPU, NCCL send/recv of the halos and an NCCL max-reduction of the signal
    speed.  Needs two GPUs (skipped otherwise); bit-equality with the undivided grid."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    import torch.multiprocessing as mp
    cspt, slab = mods
    nz, world = 26, 2
    out = str(tmp_path / "slab")
    mp.spawn(_nccl_rank, args=(world, 29533, nz, out), nprocs=world, join=True)
    w = wl.random_smooth(40, 12, nz, bc=(P, P, P, P, P, P))
    one = cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, cspt.F64)
    one.set_state(*w.fields())
    dts = [one.step_cfl(w.cfl, want_dt=True) for _ in range(7)]
    ref = torch.stack(one.get_conserved()).cpu()
    for r in range(world):
        d = torch.load("%s.%d" % (out, r))
        assert d["dts"][:6] == dts[:6]
        assert torch.equal(d["U"], ref[:, d["z0"]:d["z1"]])
    one.close()


def test_slabs_fp32_and_disk_vacuum(mods):
    cspt, slab = mods
    w = wl.disk(n=32)
    _, a, b, _ = _run_both(cspt, slab, w, 4, 6)
    for q in range(5):
        assert np.array_equal(a[q], b[q]), q
    assert np.isfinite(b[0]).all()


def test_slabs_match_the_oracle(mods, oracle_mod):
    cspt, slab = mods
    w = wl.random_smooth(24, 20, 32, bc=(O, O, P, P, P, P))
    f, _, b, dts = _run_both(cspt, slab, w, 2, 10)
    o = make_oracle(oracle_mod, w)
    o.set_state(*f)
    for n, dt in enumerate(dts):
        # bit-exact on the same input state; later states agree to round-off only, and so do their CFL steps
        assert o.compute_dt(w.cfl) == dt if n == 0 else abs(o.compute_dt(w.cfl) / dt - 1.0) < 1e-12
        o.step(dt)
    errs = field_errors(b, o.get_conserved())
    assert max(errs) < 1e-11, errs


def test_slab_protocol_errors(mods):
    cspt, slab = mods
    w = wl.random_smooth(16, 8, 8)
    bc = slab.slab_bc(w.bc, 0, 2)
    s = cspt.Solver(w.nx, w.ny, 8, w.h, w.gamma, bc, cspt.F64)
    f = w.fields()
    with pytest.raises(cspt.CsptError) as e:
        s.fill_ghosts()                                  # no state yet
    assert e.value.code == cspt.ESTATE
    s.set_state(*f)
    with pytest.raises(cspt.CsptError) as e:
        s.step_filled(1e-3)                              # psi halo not exchanged, f not formed
    assert e.value.code == cspt.ESTATE
    s.halo_put(4, s.halo_get(5, cspt.HALO_PSI), cspt.HALO_PSI)
    s.halo_put(5, s.halo_get(4, cspt.HALO_PSI), cspt.HALO_PSI)
    s.finish_state()
    for call in (lambda: s.step(1e-3), lambda: s.step_cfl(0.4), lambda: s.run_cfl(0.4, 2)):
        with pytest.raises(cspt.CsptError) as e:
            call()                                       # a slab cannot fill its EXTERNAL faces by itself
        assert e.value.code == cspt.ESTATE
    # cspt_step_filled refuses ghost layers that belong to an earlier state: it wants cspt_fill_ghosts and
    # one cspt_halo_put(CSPT_HALO_U) per EXTERNAL face since the state last changed
    def stale(call):
        with pytest.raises(cspt.CsptError) as e:
            call()
        assert e.value.code == cspt.ESTATE
    stale(lambda: s.step_filled(1e-3))                   # nothing filled yet
    s.fill_ghosts()
    stale(lambda: s.step_filled(1e-3))                   # no halos
    s.halo_put(4, s.halo_get(5))
    stale(lambda: s.step_filled(1e-3))                   # one face only
    s.halo_put(5, s.halo_get(4))
    s.step_filled(1e-3)                                  # complete: runs
    stale(lambda: s.step_filled(1e-3))                   # the new state has no ghost layers
    s.fill_ghosts()
    s.halo_put(4, s.halo_get(5))
    s.halo_put(5, s.halo_get(4))
    s.set_conserved(*s.get_conserved())                  # the state changed under the halos
    stale(lambda: s.step_filled(1e-3))
    with pytest.raises(cspt.CsptError):
        cspt.Solver(8, 8, 8, 0.1, 1.4, (cspt.BC_EXTERNAL, cspt.BC_EXTERNAL, 0, 0, 0, 0), cspt.F64)   # z faces only
    plain = cspt.Solver(8, 8, 8, 0.1, 1.4, (0,) * 6, cspt.F64)
    plain.set_state(*wl.random_smooth(8, 8, 8).fields())
    stale(lambda: plain.step_filled(1e-3))               # also on a ctx without EXTERNAL faces
    plain.fill_ghosts()
    plain.step_filled(1e-3)
    with pytest.raises(cspt.CsptError) as e:
        plain.halo_put(4, plain.halo_get(5))             # face is not EXTERNAL
    assert e.value.code == cspt.EINVAL
    s.close()
    plain.close()
