"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by
element, on the same seeded inputs.  Tolerances (BASELINE.json north_star; DESIGN.md
section 6): fp64 1e-11 normwise per conserved field after 10 steps, fp32 1e-4 against
the fp64 oracle started from the fp32-rounded inputs with the same dt sequence (G22);
CFL dt and vacuum mask bit-exact on the same input state.
"""
import math

import numpy as np
import pytest

from oracle_util import g9_threshold_state, make_oracle, run_to
from paper_1912_04855_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL64 = 1e-11
TOL32 = 1e-4


@pytest.fixture(scope="module")
def cspt():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1912_04855_b200 import build, cspt as mod
    build.build()
    mod.lib()          # fails loudly if libcspt.so is missing
    return mod


def make_solver(cspt, w, dtype=None):
    d = cspt.F64 if (dtype or w.dtype) == "f64" else cspt.F32
    return cspt.Solver(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, d)


def field_errors(gpu, orc):
    """Normwise max error per conserved field (G21).  A momentum component that vanishes
    identically in the oracle is measured against the momentum scale sqrt(rho E)."""
    gpu = [np.asarray(a, dtype=np.float64) for a in gpu]
    orc = [np.asarray(a, dtype=np.float64) for a in orc]
    mscale = math.sqrt(float(np.max(np.abs(orc[0]))) * float(np.max(np.abs(orc[4]))))
    errs = []
    for q in range(5):
        den = float(np.max(np.abs(orc[q])))
        if 1 <= q <= 3 and den < 1e-6 * mscale:
            den = mscale
        errs.append(float(np.max(np.abs(gpu[q] - orc[q]))) / max(den, 1e-300))
    return errs


def run_pair(cspt, orc_mod, w, steps, tol, gpu_dtype=None, fields=None, check_dt=True, limiter=0, kernel=0, riemann=0):
    """Steps both sides with the oracle's dt sequence; returns (solver, oracle)."""
    f = fields if fields is not None else w.fields()
    gd = gpu_dtype or w.dtype
    o = make_oracle(orc_mod, w, dtype="f64" if gd == "f32" else w.dtype)
    if kernel:
        o.set_kernel(kernel)
    o.set_state(*[np.asarray(a, dtype=np.float64) for a in f] if gd == "f32" else f)
    s = make_solver(cspt, w, dtype=gd)
    if kernel:
        s.set_kernel(kernel)       # before set_state: f = -D[psi] uses the kernel's lattice weights
    s.set_state(*f)
    if limiter:
        o.set_limiter(limiter)
        s.set_limiter(limiter)
    if riemann:
        o.set_riemann(riemann)
        s.set_riemann(riemann)
    if check_dt and gd == "f64":
        assert s.compute_dt(w.cfl) == o.compute_dt(w.cfl)          # bit-exact on the same input
    for n in range(steps):
        dt = o.compute_dt(w.cfl)
        if gd == "f32":
            dt = float(np.float32(dt))
        o.step(dt)
        s.step(dt)
    got = [t.cpu().numpy() for t in s.get_conserved()]
    errs = field_errors(got, o.get_conserved())
    assert all(np.isfinite(a).all() for a in got)
    assert max(errs) < tol, errs
    return s, o


# ---- element-by-element, several tiles and a ragged tail, every boundary kind -----------------
@pytest.mark.parametrize("dims,bc", [
    ((40, 37, 21), [0] * 6),
    ((33, 18, 45), [1] * 6),
    ((24, 20, 19), [2, 1, 0, 0, 1, 1]),
    ((17, 5, 4), [1, 2, 2, 1, 0, 0]),
    ((5, 1, 3), [0] * 6),
    ((70, 19, 150), [1, 1, 0, 0, 2, 1]),      # several z chunks (capped at 64 planes), ragged x / y tiles
])
def test_random_smooth_fp64(cspt, oracle_mod, dims, bc):
    w = wl.random_smooth(*dims, bc=bc)
    run_pair(cspt, oracle_mod, w, 10, TOL64)


def test_random_smooth_fp32(cspt, oracle_mod):
    w = wl.random_smooth(40, 37, 21, dtype="f32")
    run_pair(cspt, oracle_mod, w, 10, TOL32)
    # and the fp32 GPU path against the fp32 oracle instance: same arithmetic type
    o32 = make_oracle(oracle_mod, w)
    s = make_solver(cspt, w)
    f = w.fields()
    o32.set_state(*f)
    s.set_state(*f)
    assert np.float32(s.compute_dt(w.cfl)) == np.float32(o32.compute_dt(w.cfl))     # bit-exact in fp32 too


# ---- the five BASELINE.json configs at sizes the oracle finishes in seconds ------------------------
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_cfg1_sod(cspt, oracle_mod, axis):
    w = wl.sod(axis=axis)
    run_pair(cspt, oracle_mod, w, 10, TOL64)


def test_cfg1_sod_full_run_vs_exact(cspt, oracle_mod):
    """The whole config-1 run with the GPU's own compute_dt: 70 steps to t = 0.2, compared with the
    exact Riemann solution to the same L1 bound the oracle is pinned to."""
    import exact_riemann as er
    w = wl.sod()
    s = make_solver(cspt, w)
    s.set_state(*w.fields())
    t, n = 0.0, 0
    while t < w.t_end * (1 - 1e-14):
        dt = min(s.compute_dt(w.cfl), w.t_end - t)
        s.step(dt)
        t += dt
        n += 1
    rho = s.get_state()[0].cpu().numpy()[0, 0, :]
    x = (np.arange(w.nx) + 0.5) / w.nx
    re, _, _ = er.sample((x - 0.5) / w.t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    assert n == 70
    assert float(np.mean(np.abs(rho - re))) < 1.3e-2
    o = make_oracle(oracle_mod, w)
    o.set_state(*w.fields())
    run_to(o, w.cfl, t_end=w.t_end)
    assert np.max(np.abs(rho - o.get_state()[0][0, 0, :])) < 1e-9       # 70 steps through a shock


def test_cfg2_sedov(cspt, oracle_mod):
    run_pair(cspt, oracle_mod, wl.sedov(n=28), 10, TOL64)


@pytest.mark.parametrize("variant", ["flow", "gamma2", "isothermal"])
def test_cfg3_well(cspt, oracle_mod, variant):
    w = wl.well(n=28, variant=variant)
    s, o = run_pair(cspt, oracle_mod, w, 10, TOL64)
    if variant == "gamma2":      # well-balanced: the GPU path keeps the exact discrete equilibrium too
        rho, u, v, ww, p = [t.cpu().numpy() for t in s.get_state()]
        assert max(np.max(np.abs(a)) for a in (u, v, ww)) < 1e-13


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_cfg4_turbulence(cspt, oracle_mod, dtype):
    w = wl.turbulence(n=32, dtype=dtype)
    run_pair(cspt, oracle_mod, w, 10, TOL64 if dtype == "f64" else TOL32)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_cfg5_disk_vacuum(cspt, oracle_mod, dtype):
    w = wl.disk(n=40, dtype=dtype)
    s, o = run_pair(cspt, oracle_mod, w, 10, TOL64 if dtype == "f64" else TOL32)
    # vacuum mask: bit-exact on the same state (push the oracle's state through the GPU getters)
    o_state = o.get_conserved()
    s.set_conserved(*[a.astype(np.float32 if dtype == "f32" else np.float64) for a in o_state])
    if dtype == "f64":
        assert np.array_equal(s.get_vacuum_mask().cpu().numpy(), o.get_vacuum_mask())
        assert s.compute_dt(w.cfl) == o.compute_dt(w.cfl)
        for a, b in zip(s.get_state(), o.get_state()):
            assert np.array_equal(a.cpu().numpy(), b)            # primitives use exactly rounded operations
    m = s.get_vacuum_mask().cpu().numpy()
    assert 0 < m.sum() < m.size                                  # the case really has gas and vacuum


# ---- the limiter switch: van Leer on both sides --------------------------------------
@pytest.mark.parametrize("dims,bc,dtype", [
    ((40, 37, 21), [0] * 6, "f64"),
    ((33, 18, 45), [1, 2, 0, 0, 1, 1], "f64"),
    ((40, 37, 21), [0] * 6, "f32"),
])
def test_vanleer_random_smooth(cspt, oracle_mod, dims, bc, dtype):
    w = wl.random_smooth(*dims, bc=bc, dtype=dtype)
    run_pair(cspt, oracle_mod, w, 10, TOL64 if dtype == "f64" else TOL32, limiter=cspt.LIMITER_VANLEER)


def test_vanleer_sod_and_disk(cspt, oracle_mod):
    run_pair(cspt, oracle_mod, wl.sod(axis=1), 10, TOL64, limiter=cspt.LIMITER_VANLEER)
    run_pair(cspt, oracle_mod, wl.disk(n=40, dtype="f64"), 10, TOL64, limiter=cspt.LIMITER_VANLEER)


def test_limiter_switch_changes_the_result_and_rejects_unknown_values(cspt, oracle_mod):
    import torch
    w = wl.random_smooth(20, 12, 9)
    a, b = make_solver(cspt, w), make_solver(cspt, w)
    a.set_state(*w.fields())
    b.set_state(*w.fields())
    b.set_limiter(cspt.LIMITER_VANLEER)
    a.step(1e-3)
    b.step(1e-3)
    assert not torch.equal(a.get_conserved()[0], b.get_conserved()[0])
    b.set_limiter(cspt.LIMITER_MINMOD)
    with pytest.raises(cspt.CsptError) as e:
        b.set_limiter(7)
    assert e.value.code == cspt.EINVAL


# ---- the Riemann-solver switch: LF and HLLC on both sides ----------------------------
def _fast(w):
    """The generic smooth state with three times the velocity: faces where u^L and u^R differ in sign (colliding
    and diverging streams), which is where the three solvers differ."""
    rho, u, v, ww, p, psi = w.fields()
    return (rho, 3 * u, 3 * v, 3 * ww, p, psi)


@pytest.mark.parametrize("riemann", [1, 2])
@pytest.mark.parametrize("dims,bc,dtype", [
    ((40, 37, 21), [0] * 6, "f64"),
    ((33, 18, 45), [1, 2, 0, 0, 1, 1], "f64"),
    ((70, 19, 150), [1, 1, 0, 0, 2, 1], "f64"),
    ((40, 37, 21), [0] * 6, "f32"),
])
def test_riemann_solvers_random_smooth(cspt, oracle_mod, riemann, dims, bc, dtype):
    w = wl.random_smooth(*dims, bc=bc, dtype=dtype)
    run_pair(cspt, oracle_mod, w, 10, TOL64 if dtype == "f64" else TOL32, fields=_fast(w), riemann=riemann)


@pytest.mark.parametrize("riemann", [1, 2])
def test_riemann_solvers_sod_disk_well(cspt, oracle_mod, riemann):
    run_pair(cspt, oracle_mod, wl.sod(axis=1), 10, TOL64, riemann=riemann)
    run_pair(cspt, oracle_mod, wl.disk(n=40, dtype="f64"), 10, TOL64, riemann=riemann, limiter=cspt.LIMITER_VANLEER)
    run_pair(cspt, oracle_mod, wl.well(n=28, variant="flow"), 10, TOL64, riemann=riemann)
    run_pair(cspt, oracle_mod, wl.disk(n=40, dtype="f32"), 10, TOL32, riemann=riemann)


def test_riemann_switch_changes_the_result_and_rejects_unknown_values(cspt, oracle_mod):
    import torch
    w = wl.random_smooth(20, 12, 9)
    out = []
    for r in (cspt.RIEMANN_HLL, cspt.RIEMANN_LF, cspt.RIEMANN_HLLC):
        s = make_solver(cspt, w)
        s.set_state(*_fast(w))
        s.set_riemann(r)
        for _ in range(3):
            s.step(2e-3)
        out.append(s.get_conserved()[0])
    assert not torch.equal(out[0], out[1]) and not torch.equal(out[0], out[2]) and not torch.equal(out[1], out[2])
    with pytest.raises(cspt.CsptError) as e:
        s.set_riemann(3)
    assert e.value.code == cspt.EINVAL


# ---- the smoothing-kernel switch: W ~ (1 - q^2/4)^5 on both sides ------------------------
@pytest.mark.parametrize("dims,bc,dtype", [
    ((40, 37, 21), [0] * 6, "f64"),
    ((33, 18, 45), [1, 2, 0, 0, 1, 1], "f64"),
    ((40, 37, 21), [0] * 6, "f32"),
])
def test_poly5_kernel_random_smooth(cspt, oracle_mod, dims, bc, dtype):
    w = wl.random_smooth(*dims, bc=bc, dtype=dtype)
    run_pair(cspt, oracle_mod, w, 10, TOL64 if dtype == "f64" else TOL32, kernel=cspt.KERNEL_POLY5)


def test_poly5_kernel_sod_well_disk(cspt, oracle_mod):
    run_pair(cspt, oracle_mod, wl.sod(axis=2), 10, TOL64, kernel=cspt.KERNEL_POLY5)
    run_pair(cspt, oracle_mod, wl.well(n=28, variant="flow"), 10, TOL64, kernel=cspt.KERNEL_POLY5,
             limiter=cspt.LIMITER_VANLEER)
    run_pair(cspt, oracle_mod, wl.disk(n=40, dtype="f64"), 10, TOL64, kernel=cspt.KERNEL_POLY5)


def test_kernel_switch_discards_the_state_and_rejects_unknown_values(cspt, oracle_mod):
    w = wl.random_smooth(20, 12, 9)
    s = make_solver(cspt, w)
    s.set_state(*w.fields())
    s.set_kernel(cspt.KERNEL_CUBIC_SPLINE)          # unchanged: the state stays
    s.step(1e-3)
    s.set_kernel(cspt.KERNEL_POLY5)                 # changed: f = -D[psi] is stale, the state is discarded
    with pytest.raises(cspt.CsptError) as e:
        s.step(1e-3)
    assert e.value.code == cspt.ESTATE
    with pytest.raises(cspt.CsptError) as e:
        s.set_kernel(5)
    assert e.value.code == cspt.EINVAL


# ---- degenerate cases ---------------------------------------------------------------------------
def test_vacuum_shortcuts_are_exact(cspt, oracle_mod):
    """The fp32 Euler stage exists with and without the gas-vacuum shortcuts (chosen by a host-side hint from
    cspt_set_state); both must give the same bits, on a workload with vacuum and on one without."""
    for w in (wl.disk(n=48), wl.random_smooth(40, 24, 20, dtype="f32")):
        got = []
        for force in (0, 1):
            s = make_solver(cspt, w)
            s.debug_force_vacuum_variant(force)
            s.set_state(*w.fields())
            s.run_cfl(w.cfl, 6)
            s.step_cfl(w.cfl)
            got.append([t.cpu().numpy() for t in s.get_conserved()])
            s.close()
        for a, b in zip(*got):
            assert np.array_equal(a, b)
        hinted = make_solver(cspt, w)                    # no override: the hint picks one of the two
        hinted.set_state(*w.fields())
        hinted.run_cfl(w.cfl, 6)
        hinted.step_cfl(w.cfl)
        for a, b in zip(got[0], [t.cpu().numpy() for t in hinted.get_conserved()]):
            assert np.array_equal(a, b)
        hinted.close()


def test_all_vacuum_grid(cspt, oracle_mod):
    import torch
    z = np.zeros((4, 4, 8))
    s = cspt.Solver(8, 4, 4, 0.1, 1.4, [1] * 6)
    s.set_state(z, z, z, z, z, z)
    assert s.compute_dt(0.4) == float("inf")
    assert s.get_vacuum_mask().min().item() == 1
    s.step_cfl(0.4)              # dt = +inf on the device: identity step, no NaN
    assert all(torch.equal(t, torch.zeros_like(t)) for t in s.get_conserved())


def test_single_cell_and_thin_grids(cspt, oracle_mod):
    for dims in [(1, 1, 1), (2, 1, 1), (1, 7, 1)]:
        w = wl.random_smooth(*dims)
        run_pair(cspt, oracle_mod, w, 3, TOL64)


def test_step_cfl_matches_compute_dt_then_step(cspt, oracle_mod):
    import torch
    w = wl.random_smooth(20, 12, 9)
    a, b = make_solver(cspt, w), make_solver(cspt, w)
    a.set_state(*w.fields())
    b.set_state(*w.fields())
    for _ in range(4):
        dt = a.compute_dt(w.cfl)
        a.step(dt)
        assert b.step_cfl(w.cfl, want_dt=True) == dt
    for x, y in zip(a.get_conserved(), b.get_conserved()):
        assert torch.equal(x, y)


@pytest.mark.parametrize("dtype,nsteps", [("f64", 7), ("f64", 2), ("f32", 5), ("f64", 1), ("f64", 0)])
def test_run_cfl_graph_is_bit_identical_to_a_step_cfl_loop(cspt, oracle_mod, dtype, nsteps):
    """cspt_run_cfl replays two-step CUDA graphs (+ one plain step when nsteps is odd): same kernels, same
    order, so the state equals a loop of cspt_step_cfl bit for bit and the device-side time is the sum of its dt."""
    import torch
    w = wl.random_smooth(33, 18, 45, bc=[1, 2, 0, 0, 1, 1], dtype=dtype)
    a, b = make_solver(cspt, w), make_solver(cspt, w)
    a.set_state(*w.fields())
    b.set_state(*w.fields())
    t = 0.0
    for _ in range(nsteps):
        t += b.step_cfl(w.cfl, want_dt=True)
    got_t = a.run_cfl(w.cfl, nsteps, want_time=True)
    assert got_t == t
    for x, y in zip(a.get_conserved(), b.get_conserved()):
        assert torch.equal(x, y)
    # a second call continues from the other parity of the ping-pong and after a setter dropped the graphs
    a.set_limiter(cspt.LIMITER_VANLEER)
    b.set_limiter(cspt.LIMITER_VANLEER)
    a.run_cfl(w.cfl, 3)
    for _ in range(3):
        b.step_cfl(w.cfl)
    a.run_cfl(w.cfl, 4)
    for _ in range(4):
        b.step_cfl(w.cfl)
    for x, y in zip(a.get_conserved(), b.get_conserved()):
        assert torch.equal(x, y)
    assert a.launch_count() == b.launch_count()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_epilogue_speed_filter_keeps_dt_bit_exact(cspt, oracle_mod, dtype):
    """The Euler stage evaluates the exactly rounded CFL speed only for cells that pass a cheap filter; the
    maximum must still be the exact one: after every step the device-resident value equals a full exact pass
    over the same state (set_conserved invalidates the cached maximum), bit for bit."""
    for w in (wl.random_smooth(70, 19, 150, dtype=dtype, bc=[1, 1, 0, 0, 2, 1]), wl.disk(n=40, dtype=dtype),
              wl.sedov(n=28, dtype=dtype)):
        s = make_solver(cspt, w)
        s.set_state(*w.fields())
        for _ in range(6):
            s.step_cfl(w.cfl)
            dt_epilogue = s.compute_dt(w.cfl)
            U = s.get_conserved()
            s.set_conserved(*U)
            assert s.compute_dt(w.cfl) == dt_epilogue


@pytest.mark.parametrize("dtype,mach", [("f32", 1e3), ("f32", 3e3), ("f64", 1e5), ("f64", 3e6)])
def test_epilogue_speed_filter_cold_hypersonic_stream(cspt, oracle_mod, dtype, mach):
    """E - rho|u|^2/2 cancels in cold supersonic cells, so a filter with a fixed relative margin
    could reject the true maximum (from Mach ~ 300 in fp32).  The filter now compares a rigorous upper bound:
    the device-resident dt of step_cfl must still equal an exact pass over the same state, bit for bit."""
    nx, ny, nz = 40, 12, 9
    r = wl.random_smooth(nx, ny, nz, dtype=dtype)
    rho, u, v, w_, p, psi = [np.asarray(a, dtype=np.float64) for a in r.fields()]
    cs = math.sqrt(r.gamma)                       # p / rho ~ 1
    fields = [rho, mach * cs * (1 + 0.02 * u), 0.3 * mach * cs * v, 0.1 * mach * cs * w_, p, 0 * psi]
    fields = [a.astype(r.np_dtype) for a in fields]
    s = make_solver(cspt, r)
    s.set_state(*fields)
    for _ in range(5):
        s.step_cfl(r.cfl)
        dt_epilogue = s.compute_dt(r.cfl)
        U = s.get_conserved()
        s.set_conserved(*U)
        assert s.compute_dt(r.cfl) == dt_epilogue
        assert all(bool(np.isfinite(t.cpu().numpy()).all()) for t in U)


def test_host_entry_points_roundtrip(cspt, oracle_mod):
    import torch
    w = wl.random_smooth(20, 12, 9)
    f = [torch.from_numpy(a).pin_memory() for a in w.fields()]
    a, b = make_solver(cspt, w), make_solver(cspt, w)
    a.set_state(*w.fields())
    b.set_state_host(*f)
    a.step(1e-3)
    b.step(1e-3)
    out = [torch.empty(a.shape, dtype=torch.float64).pin_memory() for _ in range(5)]
    b.get_conserved_host(out)
    for x, y in zip(a.get_conserved(), out):
        assert torch.equal(x.cpu(), y)


def test_async_host_entry_points_match_the_blocking_ones(cspt, oracle_mod):
    """cspt_set_state_host_async / cspt_get_conserved_host_async (copy streams of their own) against the blocking calls,
    over three back-to-back states whose copies overlap: same bits, and a step in between waits for the staged result."""
    import torch
    ws = [wl.random_smooth(40, 24, 20, seed=s0) for s0 in (3, 4, 5)]
    w = ws[0]
    fields = [[torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in x.fields()] for x in ws]
    ref = []
    s = make_solver(cspt, w)
    for f in fields:
        out = [torch.empty((w.nz, w.ny, w.nx), dtype=torch.float64).pin_memory() for _ in range(5)]
        s.set_state_host(*f)
        s.step_cfl(w.cfl)
        s.step_cfl(w.cfl)
        s.get_conserved_host(out)
        ref.append([t.clone() for t in out])
    s.close()
    s = make_solver(cspt, w)
    outs = [[torch.empty((w.nz, w.ny, w.nx), dtype=torch.float64).pin_memory() for _ in range(5)] for _ in fields]
    for f, out in zip(fields, outs):
        s.set_state_host_async(*f)
        s.step_cfl(w.cfl)
        s.step_cfl(w.cfl)
        s.get_conserved_host_async(out)
    s.sync()
    for a, b in zip(ref, outs):
        for x, y in zip(a, b):
            assert torch.equal(x, y)
    s.close()


def test_explicit_stream_and_two_solvers_alive(cspt, oracle_mod):
    """The ctx works on the stream it was given (not only torch's current stream), and two solvers of different
    precision and size can be interleaved on their own streams."""
    import torch
    w1, w2 = wl.random_smooth(24, 20, 19), wl.random_smooth(33, 9, 12, dtype="f32")
    st1, st2 = torch.cuda.Stream(), torch.cuda.Stream()
    a = cspt.Solver(w1.nx, w1.ny, w1.nz, w1.h, w1.gamma, w1.bc, cspt.F64, stream=st1)
    b = cspt.Solver(w2.nx, w2.ny, w2.nz, w2.h, w2.gamma, w2.bc, cspt.F32, stream=st2)
    ref = make_solver(cspt, w1)
    a.set_state(*w1.fields())
    b.set_state(*w2.fields())
    ref.set_state(*w1.fields())
    for _ in range(5):
        a.step_cfl(w1.cfl)
        b.step_cfl(w2.cfl)
        ref.step_cfl(w1.cfl)
    ga, gb = a.get_conserved(), b.get_conserved()   # the binding orders its stream against torch's current one
    for x, y in zip(ga, ref.get_conserved()):
        assert torch.equal(x, y)                    # deterministic: same kernels, same result, any stream
    assert all(bool(torch.isfinite(t).all()) for t in gb)


def test_errors(cspt):
    s = cspt.Solver(8, 8, 8, 0.1, 1.4, [0] * 6)
    with pytest.raises(cspt.CsptError) as e:
        s.step(0.1)
    assert e.value.code == cspt.ESTATE
    z = np.ones((8, 8, 8))
    s.set_state(z, 0 * z, 0 * z, 0 * z, z, 0 * z)
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(cspt.CsptError) as e:
            s.step(bad)
        assert e.value.code == cspt.EINVAL
    with pytest.raises(cspt.CsptError):
        s.compute_dt(0.0)


# ---- round 3: ADVICE findings ---------------------------------------------------------------------
def test_fma_probe_runs_on_the_smallest_grid(cspt):
    """The roofline probe fills the device whatever the ctx's grid (its stores wrap around the scratch): BASELINE
    config 1 (64x4x4) used to be refused, which lost `bench.py --workload sod` its line."""
    import torch
    w = wl.sod(n=64, nt=4)
    s = make_solver(cspt, w)
    s.set_state(*w.fields())
    assert s.sm_count() == torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    r = s.probe_fma_rate()
    assert r > 1e12                                      # B200: ~1.4e13 fp64 FMA/s
    for min_ms in (30.0, 80.0):
        assert 0.6 < s.probe_fma_rate(0, min_ms=min_ms) / r < 1.6
    for k in (-1, 1, 8):
        assert s.probe_fma_rate(k) > 1e11
    before = [t.clone() for t in s.get_conserved()]      # the probe's scratch is dead between steps
    s.step_cfl(w.cfl)
    big = make_solver(cspt, wl.random_smooth(96, 64, 48))
    big.set_state(*wl.random_smooth(96, 64, 48).fields())
    assert 0.6 < big.probe_fma_rate() / r < 1.6           # same rate from a ctx whose scratch holds the whole grid
    fresh = make_solver(cspt, w)
    fresh.set_state(*w.fields())
    for a, b in zip(before, fresh.get_conserved()):
        assert torch.equal(a, b)
    fresh.step_cfl(w.cfl)
    for a, b in zip(s.get_conserved(), fresh.get_conserved()):
        assert torch.equal(a, b)
    for x in (s, big, fresh):
        x.close()


def test_hll_after_another_solver_is_the_hll_of_a_fresh_ctx(cspt):
    """cspt_set_riemann(LF | HLLC) moves an fp32 ctx to the row layout of the Euler stage; selecting HLL again moves it
    back, so the bits of an HLL run do not depend on what was selected before (include/cspt.h)."""
    import torch
    for w in (wl.disk(n=40), wl.random_smooth(40, 24, 20, dtype="f32")):
        fresh = make_solver(cspt, w)
        fresh.set_state(*w.fields())
        fresh.run_cfl(w.cfl, 4)
        fresh.step_cfl(w.cfl)
        back = make_solver(cspt, w)
        back.set_riemann(cspt.RIEMANN_HLLC)
        back.set_state(*w.fields())
        back.step_cfl(w.cfl)                              # a step on the other layout, then start over with HLL
        back.set_riemann(cspt.RIEMANN_HLL)
        back.set_state(*w.fields())
        back.run_cfl(w.cfl, 4)
        back.step_cfl(w.cfl)
        for a, b in zip(fresh.get_conserved(), back.get_conserved()):
            assert torch.equal(a, b)
        fresh.close()
        back.close()


def test_vacuum_threshold_state(cspt, oracle_mod):
    """GPU twin of tests/test_oracle_round3_pins.py::test_vacuum_threshold_of_reading_g9: one cell just below and one
    just above rho_vac = 1e-12 among exact vacuum.  Mask, primitives and the CFL time step bit for bit against the
    oracle; the sub-threshold cell does not move in a step."""
    gamma, h, cfl = 1.4, 0.1, 0.4
    U, A, B, _ = g9_threshold_state(gamma=gamma)
    nz, ny, nx = U[0].shape
    zero = np.zeros_like(U[0])
    w = wl.Workload("g9", nx, ny, nz, h, gamma, [1] * 6, (0, 0, 0), cfl, None, "f64", None)
    o = make_oracle(oracle_mod, w)
    o.set_state(zero, zero, zero, zero, zero, zero)
    o.set_conserved(*U)
    s = make_solver(cspt, w)
    s.set_state(zero, zero, zero, zero, zero, zero)
    s.set_conserved(*U)
    m = s.get_vacuum_mask().cpu().numpy()
    assert np.array_equal(m, o.get_vacuum_mask()) and m[A] == 1 and m[B] == 0
    for a, b in zip(s.get_state(), o.get_state()):
        assert np.array_equal(a.cpu().numpy(), b)
    dt = s.compute_dt(cfl)
    assert dt == o.compute_dt(cfl)
    s.step(dt)
    o.step(dt)
    got = [t.cpu().numpy() for t in s.get_conserved()]
    for q in range(5):
        assert got[q][A] == U[q][A], q
    assert max(field_errors(got, o.get_conserved())) < TOL64
    s.close()


def _gas_ball(nx, ny, nz, centre, bc, radius=0.12):
    """A ball of gas at rest (rho = p = 1) in exact vacuum: it expands into the empty bricks around it."""
    h = 1.0 / nx
    z, y, x = np.meshgrid((np.arange(nz) + 0.5) * h, (np.arange(ny) + 0.5) * h, (np.arange(nx) + 0.5) * h, indexing="ij")
    r2 = (x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2
    rho = np.where(r2 < radius ** 2, 1.0, 0.0).astype(np.float32)
    zero = np.zeros_like(rho)
    w = wl.Workload("gas-ball", nx, ny, nz, h, 1.4, list(bc), (0, 0, 0), 0.4, None, "f32", None)
    return w, (rho, zero, zero, zero, rho.copy(), zero)


@pytest.mark.parametrize("case", ["disk", "ball-outflow", "ball-periodic"])
def test_tile_skip_is_exact(cspt, case):
    """CTA-level gas-vacuum shortcut (fp32): CTAs whose inputs are all exactly 0 return early.  Same bits as the full
    evaluation, on a state where gas ENTERS bricks that were empty (the map has to follow it, through the ghost layers
    of periodic faces too), by single steps and from the CUDA graph; and the shortcut really is taken."""
    import torch
    if case == "disk":
        w = wl.disk(n=128)
        f, steps = w.fields(), 12
    elif case == "ball-outflow":
        w, f = _gas_ball(128, 72, 64, (0.3, 0.28, 0.25), [1] * 6)
        steps = 60
    else:
        w, f = _gas_ball(128, 72, 64, (0.06, 0.05, 0.45), [0] * 6)       # the ball straddles two periodic faces
        steps = 60
    got, dead = [], []
    for on in (0, 1):
        s = make_solver(cspt, w)
        s.debug_tile_skip(on)
        s.set_state(*f)
        s.step_cfl(w.cfl)
        s.run_cfl(w.cfl, steps - 2)
        s.step_cfl(w.cfl)
        dead.append(s.debug_dead_ctas())
        got.append(s.get_conserved())
        if on:
            # a new state under the same graphs: the map is rebuilt, the result is that of a fresh ctx
            U0 = [t.clone() for t in got[0]]
            s.set_conserved(*U0)
            s.run_cfl(w.cfl, 4)
            again = s.get_conserved()
            ref = make_solver(cspt, w)
            ref.debug_tile_skip(0)
            ref.set_state(*f)
            ref.set_conserved(*U0)
            ref.run_cfl(w.cfl, 4)
            for a, b in zip(again, ref.get_conserved()):
                assert torch.equal(a, b)
            # calls that use the intermediate slots as staging or scratch between steps (dead CTAs rely on the zeros
            # they left there): the steps after them still give the bits of the full evaluation
            host = [torch.empty(a.shape, dtype=a.dtype).pin_memory() for a in again]
            s.get_conserved_host(host)
            for a, b in zip(again, host):
                assert torch.equal(a.cpu(), b)
            s.probe_fma_rate()
            s.run_cfl(w.cfl, 5)
            s.get_conserved_host_async(host)
            s.sync()
            s.step_cfl(w.cfl)
            s.step_cfl(w.cfl)
            ref.run_cfl(w.cfl, 7)
            for a, b in zip(s.get_conserved(), ref.get_conserved()):
                assert torch.equal(a, b)
            ref.close()
        s.close()
    for a, b in zip(*got):
        assert torch.equal(a, b)
    assert dead[0] == 0 and dead[1] > 0, dead
    rho = got[0][0]
    assert bool(torch.isfinite(rho).all()) and float((rho == 0).float().mean()) > 0.2     # vacuum is still there
