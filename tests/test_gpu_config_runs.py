"""The five BASELINE.json configs run for the number of steps they name, at FULL size, through `cspt_run_cfl` (the
call bench.py times), checked by properties that hold at any size (where the 10-step windows of
test_gpu_fullsize.py check values): the state stays finite and rho >= 0; mass, momentum and energy are conserved to
round-off where the boundaries are periodic or the gas at an outflow face is at rest (Eq. (4): the update
is a flux difference; Eq. (7): the SPH sums are pair-antisymmetric); the Gamma = 2 hydrostatic equilibrium in the
potential well survives 100 steps at 256^3 to round-off (the well-balanced property; reading G8)."""
import numpy as np
import pytest

from paper_1912_04855_b200 import workloads as wl
from test_gpu_fullsize import device_fields

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cspt():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1912_04855_b200 import build, cspt as mod
    build.build()
    mod.lib()
    return mod


def _totals(s):
    """Sums of the five conserved fields in float64."""
    return [float(t.double().sum().item()) for t in s.get_conserved()]


def _run(cspt, w, steps):
    import torch
    dev = torch.device("cuda", torch.cuda.current_device())
    s = cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, cspt.F64 if w.dtype == "f64" else cspt.F32)
    f = device_fields(w, dev)
    s.set_state(*f)
    del f
    torch.cuda.empty_cache()
    before = _totals(s)
    t = s.run_cfl(w.cfl, steps, want_time=True)
    after = _totals(s)
    U = s.get_conserved()
    assert all(bool(torch.isfinite(q).all()) for q in U), w.name
    assert float(U[0].min().item()) >= 0.0, w.name
    assert np.isfinite(t) and t > 0
    return s, before, after, U


def test_cfg2_sedov_200_steps(cspt):
    w = wl.sedov()
    s, b, a, U = _run(cspt, w, w.steps)
    # the blast has not reached the outflow faces: the gas there is at rest, every boundary flux is exactly 0
    assert abs(a[0] / b[0] - 1) < 1e-12 and abs(a[4] / b[4] - 1) < 1e-11, (b, a)
    assert float(U[0].max().item()) > 1.5                 # a shock shell has formed
    m = [float(U[q].abs().max().item()) for q in (1, 2, 3)]
    assert max(m) / min(m) - 1 < 1e-9                     # the three axes are equivalent (octant symmetry)
    s.close()


def test_cfg3_well_flow_100_steps_and_equilibrium_at_full_size(cspt):
    import torch
    w = wl.well()
    s, b, a, U = _run(cspt, w, w.steps)
    s.close()
    del U
    # companion at rest: the discrete Gamma = 2 equilibrium is preserved to round-off for 100 steps at 256^3
    w = wl.well(variant="gamma2")
    s, b, a, U = _run(cspt, w, w.steps)
    rho, u, v, ww, p = s.get_state()
    vmax = max(float(q.abs().max().item()) for q in (u, v, ww))
    rho0 = device_fields(w, rho.device)[0]
    drift = float(((rho - rho0).abs() / rho0).max().item())
    assert vmax < 1e-12 and drift < 1e-12, (vmax, drift)
    assert abs(a[0] / b[0] - 1) < 1e-13 and abs(a[4] / b[4] - 1) < 1e-13
    s.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_cfg4_turbulence_50_steps_conserves(cspt, dtype):
    w = wl.turbulence(dtype=dtype)
    s, b, a, U = _run(cspt, w, w.steps)
    tol = 1e-12 if dtype == "f64" else 2e-6
    scale_m = (b[0] * b[4]) ** 0.5
    assert abs(a[0] / b[0] - 1) < tol and abs(a[4] / b[4] - 1) < tol, (b, a)
    for q in (1, 2, 3):
        assert abs(a[q] - b[q]) / scale_m < tol, (q, b, a)
    s.close()


def test_cfg5_disk_20_steps(cspt):
    w = wl.disk()
    s, b, a, U = _run(cspt, w, w.steps)
    # the gas stays far from the outflow faces: mass is conserved to fp32 round-off
    assert abs(a[0] / b[0] - 1) < 2e-6, (b, a)
    mask = s.get_vacuum_mask()
    frac = float(mask.float().mean().item())
    assert 0.5 < frac < 0.95, frac                       # most of the box is, and stays, vacuum
    s.close()
