"""Round-3 pins of the oracle (CPU): the two places the round-2 review could still break without failing a pin.

1. The time-centring of the particle velocity in Eq. (5), (6): xi* = dt (u^n + u*)/2 and
   xi^{n+1} = xi*/2 + dt (u^n + u~)/4.  These are Heun's rule for dr/dt = u, which integrates a CONSTANT acceleration
   exactly: for uniform gas in psi = g x both offsets equal the ballistic displacement u^n dt - g dt^2/2 to round-off.
   A mistake here (dt u*, or dt u~/2 in place of the average) sits inside the scheme's truncation error, so no order
   or invariant test sees it; the offsets themselves do (read through the hook orc_get_offsets).
2. The vacuum threshold of reading G9 (rho <= rho_vac = 1e-12 is vacuum: u = p = 0, no signal speed, no face
   velocity), on a state that holds a cell just below and a cell just above the threshold.
"""
import math

import numpy as np

from oracle_util import g9_threshold_state, make_oracle
from paper_1912_04855_b200 import workloads as wl


def _oracle(orc, nx, ny, nz, h, gamma, bc):
    w = wl.Workload("custom", nx, ny, nz, h, gamma, bc, (0, 0, 0), 0.4, None, "f64", None)
    return make_oracle(orc, w)


def test_offsets_of_eq_5_and_6_are_ballistic_in_uniform_free_fall(oracle_mod):
    nx, ny, nz, h, g, gamma = 16, 6, 5, 1 / 16, 0.7, 1.4
    u0 = (0.3, -0.2, 0.1)
    z, y, x = np.meshgrid((np.arange(nz) + 0.5) * h, (np.arange(ny) + 0.5) * h, (np.arange(nx) + 0.5) * h, indexing="ij")
    one = np.ones_like(x)
    o = _oracle(oracle_mod, nx, ny, nz, h, gamma, [1, 1, 0, 0, 0, 0])
    o.set_state(2 * one, u0[0] * one, u0[1] * one, u0[2] * one, one, g * x)
    dt = 0.4 * o.compute_dt(0.4)
    o.step(dt)
    inner = (slice(3, 3 + nz), slice(3, 3 + ny), slice(3, 3 + nx))
    for which in (0, 1):                                  # xi* of Eq. (5), xi^{n+1} of Eq. (6)
        want = (u0[0] * dt - 0.5 * g * dt * dt, u0[1] * dt, u0[2] * dt)
        for d in range(3):
            got = o.get_offsets(which, d)[inner]
            assert np.max(np.abs(got - want[d])) < 1e-15, (which, d, float(np.max(np.abs(got - want[d]))))
    # the two mistakes the pin is there for are far outside that bound
    assert abs((u0[0] - g * dt) * dt - want[0]) > 1e-6            # xi* = dt u*
    assert abs(0.25 * g * dt * dt) > 1e-6                         # xi = xi*/2 + dt u~/2
    # and the gas itself fell freely: u = u0 - g dt, uniform
    rho, u, v, w, p = o.get_state()
    assert np.max(np.abs(u - (u0[0] - g * dt))) < 1e-14 and np.max(np.abs(v - u0[1])) < 1e-15
    o.close()


def test_vacuum_threshold_of_reading_g9(oracle_mod):
    gamma, h, cfl = 1.4, 0.1, 0.4
    U, A, B, (rho_b, u_b, p_b) = g9_threshold_state(gamma=gamma)
    nz, ny, nx = U[0].shape
    o = _oracle(oracle_mod, nx, ny, nz, h, gamma, [1] * 6)
    zero = np.zeros_like(U[0])
    o.set_state(zero, zero, zero, zero, zero, zero)
    o.set_conserved(*U)
    # mask: 1 at and below rho_vac (A and the exact vacuum), 0 above (B)
    mask = o.get_vacuum_mask()
    assert mask[A] == 1 and mask[B] == 0 and int(mask.sum()) == mask.size - 1
    # primitives: a vacuum cell has no velocity and no pressure although m / rho = 2e9 there
    rho, u, v, w, p = o.get_state()
    assert rho[A] == 5e-13 and u[A] == 0 and v[A] == 0 and w[A] == 0 and p[A] == 0
    assert abs(u[B] - u_b) < 1e-15 and abs(p[B] / p_b - 1) < 1e-12 and v[B] == 0
    # CFL: only B counts (c + |u| of B), not the 2e9 of the sub-threshold cell
    want_dt = cfl * h / (math.sqrt(gamma * p_b / rho_b) + u_b)
    dt = o.compute_dt(cfl)
    assert abs(dt / want_dt - 1) < 1e-12, (dt, want_dt)
    # one step: the sub-threshold cell among exact vacuum does not move (no pressure, no face velocity)
    o.step(dt)
    after = o.get_conserved()
    for q in range(5):
        assert after[q][A] == U[q][A], q
    # while the gas cell above the threshold does spread into its neighbours
    assert after[0][B] < U[0][B] and after[0][B[0], B[1], B[2] + 1] > 0
    o.close()
