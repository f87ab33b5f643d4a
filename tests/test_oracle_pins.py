"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types the oracle's formulas: each compares the oracle with an
independent statement -- an exact Riemann solver, a closed form, an invariant
(conservation, symmetry, equilibrium), a brute-force all-pairs evaluation of
Eq. (7) from the textbook kernel W by numerical differentiation, or a value the
paper prints (tests/golden/).  CPU only (`-m "not gpu"`).
"""
import math
import os

import numpy as np
import pytest

import exact_riemann as er
from oracle_util import make_oracle, run_to
from paper_1912_04855_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                out[k.strip()] = float(v)
    return out


def _custom(nx, ny, nz, h, gamma, bc, fields, orc, dtype="f64"):
    w = wl.Workload("custom", nx, ny, nz, h, gamma, bc, (0, 0, 0), 0.4, None, dtype, None)
    o = make_oracle(orc, w)
    o.set_state(*fields)
    return o


# ---- Eq. (7) against the textbook kernel, all pairs, numerical gradient -------
def _W_m4(r, h):
    """Monaghan M4 cubic spline, textbook form (ref. [10]); constant factor irrelevant."""
    q = r / h
    return np.where(q < 1, 1 - 1.5 * q ** 2 + 0.75 * q ** 3, np.where(q < 2, 0.25 * (2 - q) ** 3, 0.0))


def _W_poly5(r, h):
    """W ~ (1 - q^2/4)^5 on q < 2 (the square-root-free alternative)."""
    q = r / h
    return np.where(q < 2, (1 - 0.25 * q ** 2) ** 5, 0.0)


def _gradW(d, h, W=_W_m4):
    """grad_i W(|r_i - r_j|) by central differences of the textbook W (d = r_i - r_j)."""
    eps = 1e-6 * h
    g = np.zeros(3)
    for a in range(3):
        e = np.zeros(3)
        e[a] = eps
        g[a] = (W(np.linalg.norm(d + e), h) - W(np.linalg.norm(d - e), h)) / (2 * eps)
    return g


@pytest.mark.parametrize("kernel", [0, 1])
def test_Q_brute_force_all_pairs(oracle_mod, kernel):
    """PAPER.md:66 Eq. (7) on a 4^3 periodic box: every pair (i,i') with minimum-image
    lattice offset in {-1,0,1}^3, displaced particles, grad W differentiated numerically
    from the textbook spline, normalised so that the undisplaced operator differentiates
    a linear field exactly (reading G5).  Signs per reading G1."""
    n, h, gamma = 4, 0.25, 1.4
    rng = np.random.default_rng(7)
    shape = (n, n, n)
    rho = 1 + 0.3 * rng.random(shape)
    u, v, w = (0.4 * (rng.random(shape) - 0.5) for _ in range(3))
    p = 1 + 0.5 * rng.random(shape)
    psi = 0.3 * rng.random(shape)
    xi = [0.3 * h * (rng.random(shape) - 0.5) for _ in range(3)]
    o = _custom(n, n, n, h, gamma, [0] * 6, (rho, u, v, w, p, psi), oracle_mod)
    o.set_kernel(kernel)
    W = _W_m4 if kernel == 0 else _W_poly5
    Q = o.eval_Q(xi)
    fx, fy, fz = o.eval_force()

    # normalisation: raw operator applied to the field q = x on the undisplaced lattice
    offs = [(ox, oy, oz) for oz in (-1, 0, 1) for oy in (-1, 0, 1) for ox in (-1, 0, 1) if (ox, oy, oz) != (0, 0, 0)]
    c = 0.0
    for (ox, oy, oz) in offs:
        d = -h * np.array([ox, oy, oz], float)
        c += (ox * h) * _gradW(d, h, W)[0]      # SPH gradient of q = x: sum_j q_j grad_i W
    norm = 1.0 / c

    phi = np.sqrt(2 * p)
    vel = np.stack([u, v, w], -1)
    xiv = np.stack(xi, -1)
    f = np.stack([fx, fy, fz], -1)
    Qm = np.zeros(shape + (3,))
    QE = np.zeros(shape)
    for k in range(n):
        for j in range(n):
            for i in range(n):
                sm = np.zeros(3)
                se = 0.0
                for (ox, oy, oz) in offs:
                    kk, jj, ii = (k + oz) % n, (j + oy) % n, (i + ox) % n
                    d = -h * np.array([ox, oy, oz], float) + xiv[k, j, i] - xiv[kk, jj, ii]
                    gw = _gradW(d, h, W) * norm
                    sm += phi[kk, jj, ii] * gw
                    se += phi[kk, jj, ii] * np.dot(0.5 * (vel[k, j, i] + vel[kk, jj, ii]), gw)
                Qm[k, j, i] = -phi[k, j, i] * sm + rho[k, j, i] * f[k, j, i]
                QE[k, j, i] = -phi[k, j, i] * se + rho[k, j, i] * np.dot(vel[k, j, i], f[k, j, i])
    scale = np.max(np.abs(Qm))
    for a in range(3):
        assert np.max(np.abs(Q[a] - Qm[..., a])) < 2e-7 * scale
    assert np.max(np.abs(Q[3] - QE)) < 2e-7 * np.max(np.abs(QE))


def test_lattice_operator_exact_for_linear_and_quadratic(oracle_mod):
    """f = -D[psi] (G5/G6): D differentiates linear fields exactly and,
    by the lattice's symmetry, quadratic fields too (interior cells)."""
    n, h = 8, 0.125
    z, y, x = np.meshgrid(*[(np.arange(n) + 0.5) * h] * 3, indexing="ij")
    one = np.ones_like(x)
    lin = 0.7 * x - 1.3 * y + 0.4 * z + 2.0
    o = _custom(n, n, n, h, 1.4, [1] * 6, (one, 0 * one, 0 * one, 0 * one, one, lin), oracle_mod)
    fx, fy, fz = o.eval_force()
    # odd-reflection ghosts keep a linear potential linear: exact on every cell
    assert np.max(np.abs(fx + 0.7)) < 1e-13 and np.max(np.abs(fy - 1.3)) < 1e-13 and np.max(np.abs(fz + 0.4)) < 1e-13
    quad = 0.5 * x * x - 0.8 * x * y + 0.3 * z * z + 0.2 * y * z
    o = _custom(n, n, n, h, 1.4, [1] * 6, (one, 0 * one, 0 * one, 0 * one, one, quad), oracle_mod)
    fx, fy, fz = o.eval_force()
    s = (slice(1, -1),) * 3
    assert np.max(np.abs(fx + (x - 0.8 * y))[s]) < 1e-13
    assert np.max(np.abs(fy + (-0.8 * x + 0.2 * z))[s]) < 1e-13
    assert np.max(np.abs(fz + (0.6 * z + 0.2 * y))[s]) < 1e-13
    a_f, a_e, a_c, S0p = o.lattice_constants()
    assert abs(2 * a_f + 8 * a_e + 8 * a_c - 1.0) < 1e-15          # first moment = identity
    assert a_f > a_e > a_c > 0


def test_free_fall_in_linear_potential(oracle_mod):
    """Uniform gas in psi = g x: Eq. (2),(3) give du/dt = -g, so u = -g t and the gas stays
    uniform; pins the sign of the force terms of Eq. (7) (reading G1) and rho u.f."""
    nx, h, g, gamma = 16, 1 / 16, 0.5, 1.4
    z, y, x = np.meshgrid((np.arange(4) + 0.5) * h, (np.arange(4) + 0.5) * h, (np.arange(nx) + 0.5) * h, indexing="ij")
    one = np.ones_like(x)
    bc = [1, 1, 0, 0, 0, 0]
    o = _custom(nx, 4, 4, h, gamma, bc, (2 * one, 0 * one, 0 * one, 0 * one, one, g * x), oracle_mod)
    dts = run_to(o, 0.4, steps=8)
    t = sum(dts)
    rho, u, v, w, p = o.get_state()
    assert np.max(np.abs(rho - 2)) < 1e-14
    assert np.max(np.abs(u + g * t)) < 1e-14
    assert np.max(np.abs(v)) < 1e-15 and np.max(np.abs(w)) < 1e-15
    assert np.max(np.abs(p - 1)) < 1e-13


# ---- Sod tube against the exact Riemann solution -------------------------------
def _sod_l1(orc, n, axis):
    w = wl.sod(n=n, axis=axis)
    o = make_oracle(orc, w)
    o.set_state(*w.fields())
    dts = run_to(o, w.cfl, t_end=w.t_end)
    rho, u, v, ww, p = o.get_state()
    line = [slice(0, 1)] * 3
    line[2 - axis] = slice(None)
    r1 = rho[tuple(line)].ravel()
    vel = (u, v, ww)[axis][tuple(line)].ravel()
    x = (np.arange(n) + 0.5) / n
    re, ue, pe = er.sample((x - 0.5) / w.t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    # the tube is uniform across the other two axes
    spread = [np.max(np.abs(rho - np.expand_dims(r1, tuple(a for a in range(3) if a != 2 - axis))))]
    return float(np.mean(np.abs(r1 - re))), float(np.mean(np.abs(vel - ue))), r1, len(dts), spread[0]


def test_sod_vs_exact_riemann_each_axis(oracle_mod):
    """BASELINE.json configs[0]; 'reliable solutions in the vicinity of strong shock waves'
    (PAPER.md:9).  Same answer along x, y and z (axis permutation invariance, G14)."""
    res = [_sod_l1(oracle_mod, 64, a) for a in range(3)]
    for l1r, l1u, r1, nsteps, spread in res:
        assert l1r < 1.3e-2, l1r
        assert l1u < 3.0e-2, l1u
        assert spread < 1e-14
        assert np.all(np.isfinite(r1)) and r1.min() > 0.12
    assert np.max(np.abs(res[0][2] - res[1][2])) < 1e-14
    assert np.max(np.abs(res[0][2] - res[2][2])) < 1e-14
    # plateau values of the exact solution: rho*_L = 0.42632, rho*_R = 0.26557 (Toro's test 1)
    ps, us = er.star_state(1, 0, 1, 0.125, 0, 0.1, 1.4)
    assert abs(ps - 0.30313) < 1e-5 and abs(us - 0.92745) < 1e-5
    l1_128 = _sod_l1(oracle_mod, 128, 0)[0]
    assert l1_128 < 0.7 * res[0][0]


# ---- uniform flow --------------------------------------------------------------
@pytest.mark.parametrize("bc", [[0] * 6, [1] * 6, [2, 1, 0, 0, 1, 1]])
def test_uniform_flow_preserved(oracle_mod, bc):
    shape = (6, 5, 8)
    one = np.ones(shape)
    st = (1.3 * one, 0.7 * one, -0.4 * one, 0.2 * one, 0.9 * one, 0.5 * one)
    o = _custom(8, 5, 6, 0.1, 1.4, bc, st, oracle_mod)
    run_to(o, 0.4, steps=5)
    out = o.get_state()
    for a, b in zip(out, st[:5]):
        assert np.max(np.abs(a - b)) < 4e-15


# ---- well-balanced property (reading G8) ----------------
def test_gamma2_equilibrium_to_roundoff(oracle_mod):
    w = wl.well(n=20, variant="gamma2")
    o = make_oracle(oracle_mod, w)
    f0 = w.fields()
    o.set_state(*f0)
    run_to(o, w.cfl, steps=50)
    rho, u, v, ww, p = o.get_state()
    assert max(np.max(np.abs(a)) for a in (u, v, ww)) < 1e-13
    assert np.max(np.abs(rho / f0[0] - 1)) < 1e-13
    assert np.max(np.abs(p / f0[4] - 1)) < 1e-12


def test_isothermal_equilibrium_drift_is_second_order(oracle_mod):
    """Not an exact discrete equilibrium of Eq. (7) (reading G8): the drift is
    far above round-off and falls with h."""
    drift = []
    for n in (32, 64):
        w = wl.well(n=n, variant="isothermal")
        o = make_oracle(oracle_mod, w)
        o.set_state(*w.fields())
        t_end = 0.02
        run_to(o, w.cfl, t_end=t_end)
        rho, u, v, ww, p = o.get_state()
        drift.append(max(np.max(np.abs(a)) for a in (u, v, ww)))
    assert drift[0] > 1e-6
    assert drift[1] < drift[0] / 2.5, drift


# ---- conservation --------------------------------------------------------------
def test_conservation_periodic(oracle_mod):
    w = wl.random_smooth(12, 10, 8, with_psi=False)
    o = make_oracle(oracle_mod, w)
    o.set_state(*w.fields())
    s0 = [float(np.sum(a)) for a in o.get_conserved()]
    a0 = [float(np.sum(np.abs(a))) for a in o.get_conserved()]
    run_to(o, w.cfl, steps=10)
    s1 = [float(np.sum(a)) for a in o.get_conserved()]
    for b, a, sc in zip(s0, s1, a0):
        assert abs(a - b) <= 2e-14 * sc, (a, b)


def test_energy_conserved_sedov_until_wall(oracle_mod):
    w = wl.sedov(n=24)
    o = make_oracle(oracle_mod, w)
    o.set_state(*w.fields())
    E0 = float(np.sum(o.get_conserved()[4])) * w.h ** 3
    assert abs(E0 - (1.0 + 1e-5 / 0.4 * (1 - 32 * w.h ** 3))) < 1e-12        # E=1 deposited + ambient
    run_to(o, w.cfl, steps=30)
    U = o.get_conserved()
    assert abs(float(np.sum(U[4])) * w.h ** 3 / E0 - 1) < 1e-12
    assert abs(float(np.sum(U[0])) * w.h ** 3 - 1) < 1e-12
    assert U[0].min() > 0 and np.all(np.isfinite(U[4]))
    # octant symmetry of the blast (mirror in x, y, z)
    assert np.max(np.abs(U[0] - U[0][::-1, :, :])) < 1e-12
    assert np.max(np.abs(U[0] - U[0][:, ::-1, :])) < 1e-12
    assert np.max(np.abs(U[0] - U[0][:, :, ::-1])) < 1e-12
    assert np.max(np.abs(U[1] + U[1][:, :, ::-1])) < 1e-11


# ---- symmetries ----------------------------------------------------------------
def test_axis_permutation_and_mirror(oracle_mod):
    w = wl.random_smooth(8, 10, 12)
    rho, u, v, ww, p, psi = w.fields()
    o = make_oracle(oracle_mod, w)
    o.set_state(rho, u, v, ww, p, psi)
    dts = run_to(o, w.cfl, steps=5)
    ref = o.get_conserved()
    # cyclic permutation: new x = old y, new y = old z, new z = old x  (arrays are [z,y,x])
    perm = lambda a: np.ascontiguousarray(np.transpose(a, (2, 0, 1)))     # [x,z,y] -> new [z',y',x'] = [x,z,y]
    wp = wl.Workload("perm", 10, 12, 8, w.h, w.gamma, w.bc, (0, 0, 0), 0.4, None, "f64", None)
    o2 = make_oracle(oracle_mod, wp)
    o2.set_state(perm(rho), perm(v), perm(ww), perm(u), perm(p), perm(psi))
    run_to(o2, 0.4, dts=dts)
    out = o2.get_conserved()
    for a, b in zip((out[0], out[3], out[1], out[2], out[4]), ref):        # m_x' = m_y etc.
        assert np.max(np.abs(a - perm(b))) < 1e-13
    # mirror in x
    mir = lambda a: np.ascontiguousarray(a[:, :, ::-1])
    o3 = make_oracle(oracle_mod, w)
    o3.set_state(mir(rho), -mir(u), mir(v), mir(ww), mir(p), mir(psi))
    run_to(o3, 0.4, dts=dts)
    out = o3.get_conserved()
    sign = (1, -1, 1, 1, 1)
    for a, b, s in zip(out, ref, sign):
        assert np.max(np.abs(a - s * mir(b))) < 1e-13


# ---- second order on a smooth solution (readings G12, G23) ---
def test_advected_sine_convergence(oracle_mod):
    errs = []
    for n in (64, 128, 256):
        h = 1.0 / n
        x = (np.arange(n) + 0.5) * h
        rho = (1 + 0.2 * np.sin(2 * np.pi * x)).reshape(1, 1, n)
        one = np.ones_like(rho)
        o = _custom(n, 1, 1, h, 1.4, [0] * 6, (rho, one, 0 * one, 0 * one, one, 0 * one), oracle_mod)
        run_to(o, 0.4, t_end=1.0)
        r = o.get_state()[0].ravel()
        errs.append(float(np.mean(np.abs(r - rho.ravel()))))      # exact solution: one full period
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[0] < 5e-3 and errs[2] < 4e-4, errs
    assert orders[0] > 1.6 and orders[1] > 1.75, (errs, orders)


# ---- the smoothing-kernel switch (PAPER.md:68 leaves W open, :133 "different smoothing kernels can be used";
# SURVEY 8(f) NEXT-1): W ~ (1 - q^2/4)^5, whose -W'/q needs no square root -----------------------------------
def test_poly5_kernel_lattice_constants_and_linear_exactness(oracle_mod):
    n, h = 8, 0.125
    z, y, x = np.meshgrid(*[(np.arange(n) + 0.5) * h] * 3, indexing="ij")
    one = np.ones_like(x)
    lin = 0.7 * x - 1.3 * y + 0.4 * z + 2.0
    o = _custom(n, n, n, h, 1.4, [1] * 6, (one, 0 * one, 0 * one, 0 * one, one, lin), oracle_mod)
    o.set_kernel(1)
    fx, fy, fz = o.eval_force()
    assert np.max(np.abs(fx + 0.7)) < 1e-13 and np.max(np.abs(fy - 1.3)) < 1e-13 and np.max(np.abs(fz + 0.4)) < 1e-13
    a_f, a_e, a_c, S0p = o.lattice_constants()
    g = [(1 - 0.25 * m) ** 4 for m in (1, 2, 3)]                    # closed form at |o|^2 = 1, 2, 3
    S = 2 * g[0] + 8 * g[1] + 8 * g[2]
    assert abs(S0p - S) < 1e-15 and abs(S - (2 * 0.31640625 + 8 * 0.0625 + 8 * 0.00390625)) < 1e-15
    assert max(abs(a_f - g[0] / S), abs(a_e - g[1] / S), abs(a_c - g[2] / S)) < 4e-16
    assert abs(2 * a_f + 8 * a_e + 8 * a_c - 1.0) < 1e-15


def test_poly5_kernel_equilibrium_conservation_stability(oracle_mod):
    # exact discrete Gamma = 2 equilibrium (G8 holds for any lattice weights)
    w = wl.well(n=16, variant="gamma2")
    o = make_oracle(oracle_mod, w)
    f0 = w.fields()
    o.set_state(*f0)
    o.set_kernel(1)
    run_to(o, w.cfl, steps=30)
    rho, u, v, ww, p = o.get_state()
    assert max(np.max(np.abs(a)) for a in (u, v, ww)) < 1e-13
    assert np.max(np.abs(rho / f0[0] - 1)) < 1e-13
    # conservation to round-off (pair antisymmetry does not depend on the kernel)
    w = wl.random_smooth(12, 10, 8, with_psi=False)
    o = make_oracle(oracle_mod, w)
    o.set_state(*w.fields())
    o.set_kernel(1)
    s0 = [float(np.sum(a)) for a in o.get_conserved()]
    a0 = [float(np.sum(np.abs(a))) for a in o.get_conserved()]
    run_to(o, w.cfl, steps=10)
    for b, a, sc in zip(s0, [float(np.sum(a)) for a in o.get_conserved()], a0):
        assert abs(a - b) <= 2e-14 * sc, (a, b)
    # noise at rest stays small (the kernels the survey's probe found unstable grow by orders of magnitude)
    n = 12
    rng = np.random.default_rng(3)
    shape = (n, n, n)
    rho = 1 + 1e-3 * (rng.random(shape) - 0.5)
    p = 1 + 1e-3 * (rng.random(shape) - 0.5)
    z = np.zeros(shape)
    o = _custom(n, n, n, 1.0 / n, 1.4, [0] * 6, (rho, z, z, z, p, z), oracle_mod)
    o.set_kernel(1)
    run_to(o, 0.4, steps=150)
    _, u, v, ww, _ = o.get_state()
    assert math.sqrt(float(np.mean(u * u + v * v + ww * ww))) < 3e-4


def test_poly5_kernel_sod_vs_exact_riemann(oracle_mod):
    import exact_riemann as er
    w = wl.sod()
    o = make_oracle(oracle_mod, w)
    o.set_state(*w.fields())
    o.set_kernel(1)
    run_to(o, w.cfl, t_end=w.t_end)
    rho = o.get_state()[0][0, 0, :]
    x = (np.arange(w.nx) + 0.5) / w.nx
    re, _, _ = er.sample((x - 0.5) / w.t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    assert float(np.mean(np.abs(rho - re))) < 1.5e-2


# ---- the TVD limiter switch (PAPER.md:78 "should satisfy the TVD-condition", :133 "different TVD-limiters";
# SURVEY 8(f) NEXT-1): van Leer's harmonic limiter beside minmod -----------------------------------------
def _advect(oracle_mod, n, rho, limiter, t_end=1.0):
    one = np.ones_like(rho)
    o = _custom(n, 1, 1, 1.0 / n, 1.4, [0] * 6, (rho, one, 0 * one, 0 * one, one, 0 * one), oracle_mod)
    o.set_limiter(limiter)
    run_to(o, 0.4, t_end=t_end)
    return o.get_state()[0].ravel()


def test_vanleer_second_order_and_sharper_than_minmod(oracle_mod):
    """Advected smooth profile (exact solution: translation by one period).  van Leer keeps second order
    through the extrema better than minmod: higher observed order and a several times smaller error."""
    errs = {0: [], 1: []}
    for lim in (0, 1):
        for n in (32, 64, 128):
            x = (np.arange(n) + 0.5) / n
            rho = (1 + 0.2 * np.sin(2 * np.pi * x)).reshape(1, 1, n)
            errs[lim].append(float(np.mean(np.abs(_advect(oracle_mod, n, rho, lim) - rho.ravel()))))
    order_vl = [math.log2(errs[1][i] / errs[1][i + 1]) for i in range(2)]
    assert order_vl[0] > 1.8 and order_vl[1] > 1.85, (errs, order_vl)
    assert all(errs[1][i] < 0.6 * errs[0][i] for i in range(3)), errs


@pytest.mark.parametrize("limiter", [0, 1])
def test_limiters_are_tvd_on_an_advected_square_pulse(oracle_mod, limiter):
    """TVD condition: advecting a square density pulse (u = 1, p = 1: a contact, exact solution = translation)
    creates no new extrema and does not increase the total variation."""
    n = 128
    x = (np.arange(n) + 0.5) / n
    rho = np.where((x > 0.3) & (x < 0.6), 2.0, 1.0).reshape(1, 1, n)
    r = _advect(oracle_mod, n, rho, limiter, t_end=0.5)
    tv0 = float(np.sum(np.abs(np.diff(np.r_[rho.ravel(), rho.ravel()[0]]))))
    tv1 = float(np.sum(np.abs(np.diff(np.r_[r, r[0]]))))
    assert r.min() > 1.0 - 1e-10 and r.max() < 2.0 + 1e-10
    assert tv1 <= tv0 * (1 + 1e-10)
    assert abs(r.sum() - rho.sum()) < 1e-10 * rho.sum()


def test_vanleer_is_symmetric_and_reduces_to_minmod_cases(oracle_mod):
    """With a linear profile both limiters return the exact slope, so one step of pure advection agrees to
    round-off; with a monotone profile the mirrored run is the mirror image (theta(a,b) = theta(b,a))."""
    n = 64
    x = (np.arange(n) + 0.5) / n
    one = np.ones((1, 1, n))
    ramp = (1 + 0.5 * np.sin(2 * np.pi * x) ** 2).reshape(1, 1, n)
    out = {}
    for lim in (0, 1):
        for sgn in (1, -1):
            r0 = ramp if sgn == 1 else ramp[:, :, ::-1].copy()
            o = _custom(n, 1, 1, 1.0 / n, 1.4, [0] * 6, (r0, sgn * one, 0 * one, 0 * one, one, 0 * one), oracle_mod)
            o.set_limiter(lim)
            for _ in range(5):
                o.step(0.2 / n)
            out[lim, sgn] = o.get_state()[0].ravel()
        assert np.max(np.abs(out[lim, 1] - out[lim, -1][::-1])) < 1e-14
    assert np.max(np.abs(out[0, 1] - out[1, 1])) > 1e-6          # the switch really changes the scheme


# ---- gas-vacuum boundary (Fig. 2; reading G9) -------------------
def test_vacuum_fan_closed_form(oracle_mod):
    gd = _golden("vacuum_fan.txt")
    gamma, t_end = gd["gamma"], gd["t"]
    cl = math.sqrt(gamma * gd["p_L"] / gd["rho_L"])
    x0 = gd["x_head"] + t_end * cl            # head moves left at the sound speed from x0
    l1 = []
    for n in (100, 400):
        h = 1.0 / n
        x = (np.arange(n) + 0.5) * h
        gas = (x < x0).astype(float).reshape(1, 1, n)
        o = _custom(n, 1, 1, h, gamma, [1, 1, 0, 0, 0, 0], (gas * gd["rho_L"], 0 * gas, 0 * gas, 0 * gas, gas * gd["p_L"], 0 * gas), oracle_mod)
        assert np.array_equal(o.get_vacuum_mask().ravel(), (x >= x0).astype(np.uint8))
        run_to(o, 0.4, t_end=t_end)
        rho, u, v, w, p = o.get_state()
        rho = rho.ravel()
        assert np.all(np.isfinite(rho)) and rho.min() >= 0
        re, ue = er.vacuum_fan((x - x0) / t_end, gd["rho_L"], gd["p_L"], gamma)
        l1.append(float(np.mean(np.abs(rho - re))))
        # the paper's printed value: the rarefaction head sits at x = 0.5 at t = 0.3
        head = x[np.argmax(rho < 0.995)]
        assert abs(head - gd["x_head"]) < 0.04 + 2 * h, head
        assert np.max(np.abs(rho[x < gd["x_head"] - 0.08] - 1)) < 1e-3       # undisturbed ahead of the head
    assert l1[0] < 1.5e-2 and l1[1] < 0.45 * l1[0], l1


# ---- stability at rest (M << 1; reading G5) ----------------------
def test_noise_at_rest_is_stable(oracle_mod):
    n = 12
    rng = np.random.default_rng(3)
    shape = (n, n, n)
    rho = 1 + 1e-3 * (rng.random(shape) - 0.5)
    p = 1 + 1e-3 * (rng.random(shape) - 0.5)
    z = np.zeros(shape)
    o = _custom(n, n, n, 1.0 / n, 1.4, [0] * 6, (rho, z, z, z, p, z), oracle_mod)
    run_to(o, 0.4, steps=150)
    _, u, v, w, _ = o.get_state()
    rms = math.sqrt(float(np.mean(u * u + v * v + w * w)))
    assert rms < 2e-4, rms


# ---- CFL time step and vacuum mask (reading G15, G9) --------------------------
def test_compute_dt_closed_form(oracle_mod):
    shape = (4, 4, 4)
    one = np.ones(shape)
    rho, p, gamma, h = 1.2, 0.8, 1.4, 0.05
    u = 0.3 * one
    u[1, 2, 3] = -1.7                       # the fastest cell
    o = _custom(4, 4, 4, h, gamma, [0] * 6, (rho * one, u, 0.1 * one, -0.2 * one, p * one, 0 * one), oracle_mod)
    want = 0.4 * h / (math.sqrt(gamma * p / rho) + 1.7)
    assert abs(o.compute_dt(0.4) / want - 1) < 1e-14
    # all-vacuum grid: no signal speed at all
    o = _custom(4, 4, 4, h, gamma, [0] * 6, (0 * one, 0 * one, 0 * one, 0 * one, 0 * one, 0 * one), oracle_mod)
    assert o.compute_dt(0.4) == float("inf")
    assert o.get_vacuum_mask().min() == 1


def test_fp32_instance_tracks_fp64(oracle_mod):
    w64 = wl.random_smooth(10, 9, 8, dtype="f64")
    w32 = wl.random_smooth(10, 9, 8, dtype="f32")
    f32 = w32.fields()
    o64 = make_oracle(oracle_mod, w64)
    o64.set_state(*[a.astype(np.float64) for a in f32])
    o32 = make_oracle(oracle_mod, w32)
    o32.set_state(*f32)
    dts = run_to(o64, 0.4, steps=5)
    run_to(o32, 0.4, dts=dts)
    for a, b in zip(o32.get_conserved(), o64.get_conserved()):
        assert np.max(np.abs(a - b)) < 2e-5 * np.max(np.abs(b))


# ---- the paper's own accuracy experiment (reading G23): measured, not met -----------------------
def _simple_wave_exact(x, t, gamma, amp):
    """Right-going simple (Riemann) wave from c = c0 (1 + amp sin 2 pi x), u = 2 (c - c0)/(gamma - 1), isentropic:
    every value travels along its straight characteristic x = x0 + (u + c)(x0) t (exact until the wave breaks)."""
    c0 = math.sqrt(gamma)

    def speed(x0):
        c = c0 * (1 + amp * np.sin(2 * np.pi * x0))
        return c, 2 * (c - c0) / (gamma - 1)

    x0 = x.copy()
    for _ in range(200):                       # fixed point, contraction while t |d(u+c)/dx| < 1
        c, u = speed(x0)
        x0 = x - (u + c) * t
    c, u = speed(x0)
    rho = (c / c0) ** (2 / (gamma - 1))
    return rho, u, rho ** gamma


def test_simple_wave_order_is_reported_as_measured(oracle_mod):
    """PAPER.md:94 claims approximation order 1.94 / convergence order 2.04 on the 'linear transfer of a smooth
    Riemann wave' (set-up not given).  Under the literal reading of Eq. (5)-(7) the mass row of Q is zero, so the
    compression inside a step is never felt by p* or by U^{n+1/2}: second order for div u = 0 (advected profile
    above), FIRST order in time for a compressive simple wave (reading G23).  This test measures and
    bounds that order so that the number quoted in DESIGN.md is reproducible; the paper's 1.94 stays unpinned."""
    gamma, amp, t_end = 1.4, 0.05, 0.2
    errs = []
    for n in (64, 128, 256, 512):
        h = 1.0 / n
        x = (np.arange(n) + 0.5) * h
        rho, u, p = _simple_wave_exact(x, 0.0, gamma, amp)
        sh = lambda a: a.reshape(1, 1, n)
        z = np.zeros((1, 1, n))
        o = _custom(n, 1, 1, h, gamma, [0] * 6, (sh(rho), sh(u), z, z, sh(p), z), oracle_mod)
        run_to(o, 0.4, t_end=t_end)
        re, ue, pe = _simple_wave_exact(x, t_end, gamma, amp)
        errs.append(float(np.mean(np.abs(o.get_state()[0].ravel() - re))))
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(3)]
    assert errs[0] < 5e-3 and all(errs[i + 1] < errs[i] for i in range(3)), errs      # it does converge
    assert all(0.8 < q < 1.3 for q in orders), (errs, orders)                        # at first order, not 1.94
    print("simple wave L1(rho):", errs, "orders:", orders)


def test_linear_transfer_of_a_smooth_wave_at_the_papers_resolutions(oracle_mod):
    """'linear transfer of smooth Riemann wave ... N = 400, 800, 1600, 3200, 6400 ... approximation order
    of about 1.94; order of convergence is 2.04'.  Read as LINEAR transport (the profile is carried by a uniform flow,
    exact solution = translation; reading G23 (i)) the oracle is second order on the paper's first three grids with the
    default minmod limiter (measured 1.93, 1.95) and with van Leer's limiter (2.09).  The paper gives no set-up
    (t_end = 0.125 and the amplitude 0.2 are this test's), so the closeness to the printed 1.94 is NOT a pin of the
    paper's number: this is a second-order check for div u = 0 transport, nothing more."""
    t_end, u0 = 0.125, 1.0
    found = {}
    for lim, grids in ((0, (400, 800, 1600)), (1, (400, 800))):
        errs = []
        for n in grids:
            h = 1.0 / n
            x = (np.arange(n) + 0.5) * h
            rho = (1 + 0.2 * np.sin(2 * np.pi * x)).reshape(1, 1, n)
            one = np.ones_like(rho)
            o = _custom(n, 1, 1, h, 1.4, [0] * 6, (rho, u0 * one, 0 * one, 0 * one, one, 0 * one), oracle_mod)
            o.set_limiter(lim)
            run_to(o, 0.4, t_end=t_end)
            exact = 1 + 0.2 * np.sin(2 * np.pi * (x - u0 * t_end))
            errs.append(float(np.mean(np.abs(o.get_state()[0].ravel() - exact))))
        found[lim] = [math.log2(errs[i] / errs[i + 1]) for i in range(len(grids) - 1)]
    print("linear transfer orders (minmod, van Leer):", found)
    assert all(q > 1.85 for q in found[0]), found                      # second order (the paper prints 1.94)
    assert all(1.95 < q < 2.15 for q in found[1]), found
