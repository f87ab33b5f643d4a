"""cspt_cfl_dt_noalloc against cspt_compute_dt (GPU).

Some users of the library cannot allocate device memory: a host code whose own arena took all of HBM at start-up, a
time loop in which cudaMalloc / cudaFree would stall the device, an in-situ monitor or coupled solver that only
receives pointers to the conserved fields.  They cannot build a ctx (its workspace is 28 padded fields), so the library
offers them one ctx-free call whose scratch is a fixed 512 KiB array inside the library itself, which caps the grid at
268 435 456 cells.  This file checks that the call returns what the ctx path returns -- the CFL time step is
compared BIT FOR BIT, the bar tests/test_gpu_parity.py sets for cspt_compute_dt -- on two calls in a row whose sizes
and answers differ (all calls share the scratch and find the previous call's values there), that it really takes no
device memory, and that it turns down a grid beyond its capacity.

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this side entry should not
hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import ctypes
import math

import pytest

from paper_1912_04855_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cspt():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1912_04855_b200 import build, cspt as mod
    build.build()
    mod.lib()          # fails loudly if libcspt.so is missing
    return mod


def _reference(cspt, w, steps):
    """The existing path: a ctx on workload w, advanced `steps` steps; returns (dense conserved tensors, its dt)."""
    d = cspt.F64 if w.dtype == "f64" else cspt.F32
    s = cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, d)
    s.set_state(*w.fields())
    for _ in range(steps):
        s.step_cfl(w.cfl)
    cons = [t.reshape(-1).contiguous() for t in s.get_conserved()]
    dt = s.compute_dt(w.cfl)
    s.close()
    return cons, dt


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_two_calls_in_a_row_match_compute_dt_bit_for_bit(cspt, dtype):
    import torch
    # first call: the 40^3 disk, gas and vacuum cells, 64 000 cells -> 16 slots of the scratch, the last one ragged
    # second call: fewer cells (3 slots) and slower gas, so that a slot left over from the first call, if it were
    # read, would win the maximum and shorten the time step
    wa = wl.disk(n=40, dtype=dtype)
    wb = wl.sod(n=64, nt=12, dtype=dtype)
    (ca, dta), (cb, dtb) = _reference(cspt, wa, 3), _reference(cspt, wb, 1)
    assert dta != dtb and math.isfinite(dta) and math.isfinite(dtb)
    smax_a, smax_b = wa.cfl * wa.h / dta, wb.cfl * wb.h / dtb
    assert smax_b < smax_a, "the second state must be the slower one for the stale-slot check to bite"
    tdt = torch.float64 if dtype == "f64" else torch.float32
    out = torch.full((3,), -1.0, dtype=tdt, device="cuda")
    torch.cuda.synchronize()
    free0 = None
    for rep in range(2):          # the pair twice: the very first call also looks up the scratch address
        cspt.cfl_dt_noalloc(*ca, wa.gamma, wa.h, wa.cfl, out[0:1])
        cspt.cfl_dt_noalloc(*cb, wb.gamma, wb.h, wb.cfl, out[1:2])
        torch.cuda.synchronize()
        got = out.cpu().tolist()
        assert got[0] == dta, (got[0], dta)          # bit-exact, as test_gpu_parity asks of cspt_compute_dt
        assert got[1] == dtb, (got[1], dtb)
        assert got[2] == -1.0                        # one element written per call, no more
        free = torch.cuda.mem_get_info()[0]
        if rep == 1:
            assert free == free0, "cspt_cfl_dt_noalloc took or returned device memory"
        free0 = free


def test_degenerate_sizes_and_the_capacity_limit(cspt):
    import torch
    L = cspt.lib()
    cap = cspt.noalloc_max_cells()
    assert cap == 65536 * 4096
    z = torch.zeros(5, 4096 + 7, dtype=torch.float64, device="cuda")      # all vacuum: rho = 0 everywhere
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    cspt.cfl_dt_noalloc(*z, 1.4, 0.1, 0.3, out)
    assert out.item() == math.inf
    # one gas cell at rest in the ragged tail: dt = cfl*h/c, c = sqrt(gamma p / rho), in separately rounded operations
    z[0, -1], z[4, -1] = 2.0, 5.0                                           # rho = 2, E = 5 -> p = 0.4 * 5 = 2
    cspt.cfl_dt_noalloc(*z, 1.4, 0.1, 0.3, out)
    p = (1.4 - 1.0) * 5.0
    assert out.item() == (0.3 * 0.1) / math.sqrt((1.4 * p) / 2.0)
    # no cells at all
    e = torch.zeros(0, dtype=torch.float64, device="cuda")
    cspt.cfl_dt_noalloc(e, e, e, e, e, 1.4, 0.1, 0.3, out)
    assert out.item() == math.inf
    # beyond the scratch: refused before anything is launched or read (the pointers are those of the small arrays)
    out.fill_(7.0)
    ptrs = [ctypes.c_void_p(t.data_ptr()) for t in z]
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = L.cspt_cfl_dt_noalloc(cspt.F64, cap + 1, *ptrs, 1.4, 0.1, 0.3, ctypes.c_void_p(out.data_ptr()), st)
    assert rc == cspt.ELIMIT
    assert b"capacity" in L.cspt_strerror(rc)
    torch.cuda.synchronize()
    assert out.item() == 7.0
    with pytest.raises(cspt.CsptError) as ei:
        cspt._check(rc, "cspt_cfl_dt_noalloc")
    assert ei.value.code == cspt.ELIMIT
    # argument checks
    assert L.cspt_cfl_dt_noalloc(2, 8, *ptrs, 1.4, 0.1, 0.3, ctypes.c_void_p(out.data_ptr()), st) == cspt.EINVAL
    assert L.cspt_cfl_dt_noalloc(cspt.F64, 8, *ptrs, 1.0, 0.1, 0.3, ctypes.c_void_p(out.data_ptr()), st) == cspt.EINVAL
    assert L.cspt_cfl_dt_noalloc(cspt.F64, 8, *ptrs, 1.4, 0.1, 0.3, None, st) == cspt.EINVAL
    assert L.cspt_cfl_dt_noalloc(cspt.F64, 8, None, *ptrs[1:], 1.4, 0.1, 0.3, ctypes.c_void_p(out.data_ptr()), st) == cspt.EINVAL
