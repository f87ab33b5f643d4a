"""Pins of the oracle's Riemann-solver switch ("the approximate methods of Lax-Friedrichs (LF),
Harten-Lax-van Lier (HLL), and the modified Harten-Lax-van Lier method (HLLC) [14]"; readings G13, G13b, G13c of
DESIGN.md).  The face flux the oracle used is recovered from what one step does to a piecewise-constant cold state
(no pressure: the Lagrangian stage is the identity, the limited slopes next to a single jump vanish) and compared
with the TEXTBOOK solvers written out here in their general form (with pressure arguments, p = 0 inserted
numerically), plus closed forms and invariants.  CPU only.
"""
import math

import numpy as np
import pytest

import exact_riemann as er
from oracle_util import make_oracle, run_to
from paper_1912_04855_b200 import workloads as wl

HLL, LF, HLLC = 0, 1, 2


def _custom(nx, ny, nz, h, gamma, bc, fields, orc):
    w = wl.Workload("custom", nx, ny, nz, h, gamma, bc, (0, 0, 0), 0.4, None, "f64", None)
    o = make_oracle(orc, w)
    o.set_state(*fields)
    return o


# ---- textbook solvers, general form (Toro [14], chapter 10), 1-D normal direction + two tangential velocities ----
def _prim(U):
    rho = U[0]
    vel = U[1:4] / rho
    return rho, vel


def _phys_flux(U, p, d):
    rho, vel = _prim(U)
    F = vel[d] * U.copy()
    F[1 + d] += p
    F[4] += p * vel[d]
    return F


def textbook_lf(UL, UR, pL, pR, d, a):
    return 0.5 * (_phys_flux(UL, pL, d) + _phys_flux(UR, pR, d)) - 0.5 * a * (UR - UL)


def textbook_hllc(UL, UR, pL, pR, d, SL, SR):
    """Toro (10.37)-(10.39), (10.26): wave speeds given."""
    rL, vL = _prim(UL)
    rR, vR = _prim(UR)
    uL, uR = vL[d], vR[d]
    FL, FR = _phys_flux(UL, pL, d), _phys_flux(UR, pR, d)
    if SL >= 0:
        return FL
    if SR <= 0:
        return FR
    Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))

    def star(U, r, v, u, p, S):
        fac = r * (S - u) / (S - Ss)
        out = np.empty(5)
        out[0] = fac
        out[1:4] = fac * v
        out[1 + d] = fac * Ss
        out[4] = fac * (U[4] / r + (Ss - u) * (Ss + p / (r * (S - u))))
        return out

    if Ss >= 0:
        return FL + SL * (star(UL, rL, vL, uL, pL, SL) - UL)
    return FR + SR * (star(UR, rR, vR, uR, pR, SR) - UR)


def _face_flux_from_one_step(oracle_mod, solver, d, WL, WR):
    """Cold (p = 0) piecewise-constant state with ONE jump along axis d; returns the face flux of the jump
    recovered from the change of the cell on its left: U_new = U - dt/h (F_face - u_L U_L)."""
    n, h = 12, 0.1
    dims = [3, 3, 3]
    dims[d] = n
    shape = (dims[2], dims[1], dims[0])
    idx = np.arange(n).reshape([n if a == 2 - d else 1 for a in range(3)])
    left = np.broadcast_to(idx < n // 2, shape)
    f = [np.where(left, WL[q], WR[q]).astype(float) for q in range(4)]
    zero = np.zeros(shape)
    bc = [0] * 6
    bc[2 * d] = bc[2 * d + 1] = 1
    o = _custom(dims[0], dims[1], dims[2], h, 5.0 / 3.0, bc, (f[0], f[1], f[2], f[3], zero, zero), oracle_mod)
    o.set_riemann(solver)
    U0 = [a.copy() for a in o.get_conserved()]
    dt = 0.2 * h / max(abs(WL[1 + d]), abs(WR[1 + d]), 1e-9)
    o.step(dt)
    U1 = o.get_conserved()
    cell = [1, 1, 1]
    cell[2 - d] = n // 2 - 1                                   # the cell left of the jump
    cell = tuple(cell)
    UL = np.array([U0[q][cell] for q in range(5)])
    U1c = np.array([U1[q][cell] for q in range(5)])
    UR = np.array([U0[q][tuple(c + (1 if a == 2 - d else 0) for a, c in enumerate(cell))] for q in range(5)])
    uL = WL[1 + d]
    # inflow face of that cell: uniform left state, flux u_L U_L for all three solvers when u_L > 0 ... in general the
    # face between two equal states carries F(U,U) = u U (consistency), whatever the sign
    F_in = uL * UL
    F_face = F_in - (U1c - UL) * h / dt
    return UL, UR, F_face


STATES = [
    # (rho, u, v, w) left / right
    ((3.0, 1.0, 0.3, -0.2), (1.0, -2.0, 0.1, 0.4)),        # colliding, S* > 0
    ((1.0, 0.5, -0.3, 0.2), (4.0, -1.5, 0.6, 0.1)),        # colliding, S* < 0
    ((2.0, 1.0, 0.0, 0.0), (2.0, -1.0, 0.0, 0.0)),         # symmetric collision, S* = 0
    ((1.5, -1.0, 0.2, 0.1), (0.7, 2.0, -0.1, 0.3)),        # diverging streams
    ((1.2, 2.0, 0.1, 0.2), (0.9, 0.5, 0.3, -0.4)),         # both to the right
    ((1.2, -0.5, 0.1, 0.2), (0.9, -2.5, 0.3, -0.4)),       # both to the left
]


def _rot(W, d):
    """Put the normal velocity into component d (u <-> v or w)."""
    rho, u, v, w = W
    vel = [v, w]
    out = [None, None, None]
    out[d] = u
    rest = [a for a in range(3) if a != d]
    out[rest[0]], out[rest[1]] = vel
    return (rho, out[0], out[1], out[2])


@pytest.mark.parametrize("d", [0, 1, 2])
@pytest.mark.parametrize("case", range(len(STATES)))
def test_face_flux_against_textbook_solvers(oracle_mod, d, case):
    WL, WR = _rot(STATES[case][0], d), _rot(STATES[case][1], d)
    for solver in (HLL, LF, HLLC):
        UL, UR, F = _face_flux_from_one_step(oracle_mod, solver, d, WL, WR)
        uL, uR = WL[1 + d], WR[1 + d]
        if solver == LF:
            want = textbook_lf(UL, UR, 0.0, 0.0, d, max(abs(uL), abs(uR)))
        else:
            SL, SR = min(uL, uR), max(uL, uR)
            if solver == HLL:
                # Toro (10.21) with the same wave speeds
                FL, FR = _phys_flux(UL, 0.0, d), _phys_flux(UR, 0.0, d)
                want = FL if SL >= 0 else FR if SR <= 0 else (SR * FL - SL * FR + SL * SR * (UR - UL)) / (SR - SL)
            elif uL <= uR and SL < 0 < SR:
                want = np.zeros(5)            # diverging streams: the star region is empty (0/0 in (10.37))
            else:
                want = textbook_hllc(UL, UR, 0.0, 0.0, d, SL, SR)
        scale = max(np.max(np.abs(want)), np.max(np.abs(uL * UL)), 1e-30)
        assert np.max(np.abs(F - want)) < 1e-12 * scale, (solver, d, case, F, want)


def test_hllc_mass_flux_closed_form(oracle_mod):
    """Between converging cold streams the HLLC contact moves with the mass-weighted mean velocity
    S* = (rho_L u_L + rho_R u_R)/(rho_L + rho_R) and the mass flux through the face is rho*_K S*, with
    rho*_K = rho_K (u_L - u_R)/|S_K - S*| from the jump condition across the outer wave."""
    (rL, uL, _, _), (rR, uR, _, _) = STATES[0]
    UL, UR, F = _face_flux_from_one_step(oracle_mod, HLLC, 0, STATES[0][0], STATES[0][1])
    Ss = (rL * uL + rR * uR) / (rL + rR)
    assert Ss > 0
    rs = rL * (uR - uL) / (uR - Ss)            # S_L = u_R for converging streams
    assert abs(F[0] - rs * Ss) < 1e-13
    assert abs(Ss - 0.25) < 1e-15 and abs(rs - 4.0) < 1e-14     # worked numbers for (3, 1) against (1, -2)


@pytest.mark.parametrize("solver", [LF, HLLC])
def test_uniform_flow_and_equilibrium_survive(oracle_mod, solver):
    """Consistency F(U,U) = u U (uniform flow stays uniform) and zero flux for gas at rest: the exact discrete
    Gamma = 2 equilibrium (reading G8) is kept to round-off with every solver."""
    shape = (6, 5, 8)
    one = np.ones(shape)
    st = (1.3 * one, 0.7 * one, -0.4 * one, 0.2 * one, 0.9 * one, 0.5 * one)
    o = _custom(8, 5, 6, 0.1, 1.4, [1] * 6, st, oracle_mod)
    o.set_riemann(solver)
    run_to(o, 0.4, steps=5)
    for a, b in zip(o.get_state(), st[:5]):
        assert np.max(np.abs(a - b)) < 4e-15
    w = wl.well(n=16, variant="gamma2")
    o = make_oracle(oracle_mod, w)
    f0 = w.fields()
    o.set_state(*f0)
    o.set_riemann(solver)
    run_to(o, w.cfl, steps=30)
    rho, u, v, ww, p = o.get_state()
    assert max(np.max(np.abs(a)) for a in (u, v, ww)) < 1e-13
    assert np.max(np.abs(rho / f0[0] - 1)) < 1e-13


@pytest.mark.parametrize("solver", [LF, HLLC])
def test_conservation_and_symmetry(oracle_mod, solver):
    w = wl.random_smooth(12, 10, 8, with_psi=False)
    rho, u, v, ww, p, psi = w.fields()
    o = make_oracle(oracle_mod, w)
    o.set_state(rho, 3 * u, 3 * v, 3 * ww, p, psi)           # faster flow: faces with both signs of u^L, u^R
    o.set_riemann(solver)
    s0 = [float(np.sum(a)) for a in o.get_conserved()]
    a0 = [float(np.sum(np.abs(a))) for a in o.get_conserved()]
    dts = run_to(o, w.cfl, steps=10)
    ref = o.get_conserved()
    for b, a, sc in zip(s0, [float(np.sum(a)) for a in ref], a0):
        assert abs(a - b) <= 2e-14 * sc, (a, b)
    mir = lambda a: np.ascontiguousarray(a[:, :, ::-1])
    o3 = make_oracle(oracle_mod, w)
    o3.set_state(mir(rho), -3 * mir(u), 3 * mir(v), 3 * mir(ww), mir(p), mir(psi))
    o3.set_riemann(solver)
    run_to(o3, 0.4, dts=dts)
    for a, b, s in zip(o3.get_conserved(), ref, (1, -1, 1, 1, 1)):
        assert np.max(np.abs(a - s * mir(b))) < 1e-13


def _sod(oracle_mod, solver, n=64):
    w = wl.sod(n=n)
    o = make_oracle(oracle_mod, w)
    o.set_state(*w.fields())
    o.set_riemann(solver)
    run_to(o, w.cfl, t_end=w.t_end)
    rho = o.get_state()[0][0, 0, :]
    x = (np.arange(n) + 0.5) / n
    re, _, _ = er.sample((x - 0.5) / w.t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    return float(np.mean(np.abs(rho - re))), rho


def test_sod_all_solvers(oracle_mod):
    """All three converge to the exact Riemann solution; in the Sod tube every face velocity is >= 0, where HLLC
    coincides with HLL, and LF differs only where u^L != u^R."""
    l1 = {s: _sod(oracle_mod, s) for s in (HLL, LF, HLLC)}
    for s in (HLL, LF, HLLC):
        assert l1[s][0] < 1.6e-2, (s, l1[s][0])
        assert _sod(oracle_mod, s, n=128)[0] < 0.7 * l1[s][0]
    assert np.max(np.abs(l1[HLLC][1] - l1[HLL][1])) < 1e-13
    assert np.max(np.abs(l1[LF][1] - l1[HLL][1])) > 1e-4


def test_lf_reduces_to_upwinding_and_differs_only_across_velocity_jumps(oracle_mod):
    """With a = max(|u^L|,|u^R|) (reading G13b) the Lax-Friedrichs flux is the upwind flux wherever u^L = u^R, so on
    uniform-velocity advection the three solvers coincide to round-off (and HLLC equals HLL wherever the
    streams do not collide); across a velocity gradient LF adds (a - |u|)(U^R - U^L)/2 of diffusion: a density
    pulse in a converging velocity field comes out different from HLL, but only at the O(du) level (this local LF
    is NOT the classical a = h/dt flux, which would smear the pulse and break the equilibria)."""
    n = 128
    x = (np.arange(n) + 0.5) / n
    rho = np.where((x > 0.35) & (x < 0.65), 2.0, 1.0).reshape(1, 1, n)
    one = np.ones_like(rho)
    u = (0.5 - 0.4 * np.tanh((x - 0.5) / 0.1)).reshape(1, 1, n)
    res = {}
    for s in (HLL, LF, HLLC):
        o = _custom(n, 1, 1, 1.0 / n, 1.4, [0] * 6, (rho, u, 0 * one, 0 * one, 1e-6 * one, 0 * one), oracle_mod)
        o.set_riemann(s)
        run_to(o, 0.4, t_end=0.1)
        res[s] = o.get_state()[0].ravel()
        assert np.all(np.isfinite(res[s])) and res[s].min() > 0
        assert abs(res[s].sum() - rho.sum()) < 1e-10 * rho.sum()
    dlf = float(np.mean(np.abs(res[LF] - res[HLL])))          # L1: the pulse edges move by a fraction of a cell
    assert 1e-5 < dlf < 1e-2, dlf
    assert np.max(np.abs(res[HLLC] - res[HLL])) < 1e-13          # u > 0 everywhere: no colliding face
    out = {}
    for s in (HLL, LF, HLLC):
        o = _custom(n, 1, 1, 1.0 / n, 1.4, [0] * 6, (rho, one, 0 * one, 0 * one, one, 0 * one), oracle_mod)
        o.set_riemann(s)
        run_to(o, 0.4, t_end=0.2)
        out[s] = o.get_state()[0].ravel()
    assert np.max(np.abs(out[LF] - out[HLL])) < 1e-12 and np.max(np.abs(out[HLLC] - out[HLL])) < 1e-12
