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
