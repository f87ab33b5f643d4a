"""Helpers shared by the oracle pins and the GPU parity tests (test side only)."""
import numpy as np


def make_oracle(orc, w, dtype=None):
    d = orc.F64 if (dtype or w.dtype) == "f64" else orc.F32
    o = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.gamma, w.bc, d)
    return o


def run_to(o, cfl, t_end=None, steps=None, dts=None):
    """Advance with dt = compute_dt(cfl), last step clipped to hit t_end; or a fixed
    number of steps; or a prescribed dt sequence.  Returns the dt list."""
    used = []
    if dts is not None:
        for dt in dts:
            o.step(dt)
            used.append(dt)
        return used
    t = 0.0
    while True:
        if steps is not None and len(used) >= steps:
            break
        if t_end is not None and t >= t_end * (1 - 1e-14):
            break
        dt = o.compute_dt(cfl)
        if t_end is not None and t + dt > t_end:
            dt = t_end - t
        o.step(dt)
        t += dt
        used.append(dt)
    return used


def normwise(a, b):
    """max|a-b| / max|b| (reading G21); 0 if both vanish."""
    den = float(np.max(np.abs(b)))
    num = float(np.max(np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64))))
    return 0.0 if num == 0.0 else num / max(den, 1e-300)


def g9_threshold_state(nx=10, ny=8, nz=8, gamma=1.4):
    """Conserved fields (nz, ny, nx) for the pins of reading G9 (rho_vac = 1e-12): exact vacuum everywhere except
    cell A = (i, j, k) = (3, 3, 3) just BELOW the threshold (rho = 5e-13) with large momentum and energy, and cell
    B = (7, 5, 4) just ABOVE it (rho = 2e-12, u = 0.5, p = 3e-12).  A and B are 4 cells apart (one step reaches 3).
    Input data only: none of the method's arithmetic."""
    U = [np.zeros((nz, ny, nx)) for _ in range(5)]
    A, B = (3, 3, 3), (4, 5, 7)                      # (k, j, i)
    U[0][A], U[1][A], U[2][A], U[3][A], U[4][A] = 5e-13, 1e-3, -2e-3, 5e-4, 7.0
    rho_b, u_b, p_b = 2e-12, 0.5, 3e-12
    U[0][B], U[1][B], U[4][B] = rho_b, rho_b * u_b, p_b / (gamma - 1) + 0.5 * rho_b * u_b * u_b
    return U, A, B, (rho_b, u_b, p_b)
