"""Exact solution of the 1-D Riemann problem for the ideal-gas Euler equations.

Textbook algorithm (Toro, ref. [14] of the paper): Newton iteration
on the pressure function f(p) = f_L(p) + f_R(p) + (u_R - u_L), then sampling of
the self-similar solution at xi = x/t.  Own restatement; used only to pin the
oracle (tests/test_oracle_pins.py).  Also the closed-form rarefaction fan into
vacuum.
"""
import math

import numpy as np


def _f(p, rho, pk, g):
    """Pressure function of one side and its derivative."""
    c = math.sqrt(g * pk / rho)
    if p > pk:  # shock
        A = 2.0 / ((g + 1.0) * rho)
        B = (g - 1.0) / (g + 1.0) * pk
        s = math.sqrt(A / (p + B))
        return (p - pk) * s, s * (1.0 - 0.5 * (p - pk) / (B + p))
    # rarefaction
    e = (g - 1.0) / (2.0 * g)
    return 2.0 * c / (g - 1.0) * ((p / pk) ** e - 1.0), (1.0 / (rho * c)) * (p / pk) ** (-(g + 1.0) / (2.0 * g))


def star_state(rl, ul, pl, rr, ur, pr, g):
    p = max(1e-12, 0.5 * (pl + pr))
    for _ in range(200):
        fl, dl = _f(p, rl, pl, g)
        fr, dr = _f(p, rr, pr, g)
        pn = p - (fl + fr + (ur - ul)) / (dl + dr)
        pn = max(pn, 1e-14)
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fl, _ = _f(p, rl, pl, g)
    fr, _ = _f(p, rr, pr, g)
    return p, 0.5 * (ul + ur) + 0.5 * (fr - fl)


def sample(xi, rl, ul, pl, rr, ur, pr, g):
    """(rho, u, p) at similarity coordinates xi = x/t (numpy array)."""
    ps, us = star_state(rl, ul, pl, rr, ur, pr, g)
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    gm, gp = g - 1.0, g + 1.0
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    p = np.empty_like(xi)
    for n, s in enumerate(xi):
        if s <= us:  # left of the contact
            if ps > pl:  # left shock
                sl = ul - cl * math.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
                if s <= sl:
                    r_, u_, p_ = rl, ul, pl
                else:
                    r_, u_, p_ = rl * ((ps / pl + gm / gp) / (gm / gp * ps / pl + 1.0)), us, ps
            else:  # left rarefaction
                shl = ul - cl
                cs = cl * (ps / pl) ** (gm / (2 * g))
                stl = us - cs
                if s <= shl:
                    r_, u_, p_ = rl, ul, pl
                elif s >= stl:
                    r_, u_, p_ = rl * (ps / pl) ** (1.0 / g), us, ps
                else:
                    c = 2.0 / gp * (cl + gm / 2.0 * (ul - s))
                    u_ = 2.0 / gp * (cl + gm / 2.0 * ul + s)
                    r_ = rl * (c / cl) ** (2.0 / gm)
                    p_ = pl * (c / cl) ** (2.0 * g / gm)
        else:
            if ps > pr:  # right shock
                sr = ur + cr * math.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
                if s >= sr:
                    r_, u_, p_ = rr, ur, pr
                else:
                    r_, u_, p_ = rr * ((ps / pr + gm / gp) / (gm / gp * ps / pr + 1.0)), us, ps
            else:
                shr = ur + cr
                cs = cr * (ps / pr) ** (gm / (2 * g))
                str_ = us + cs
                if s >= shr:
                    r_, u_, p_ = rr, ur, pr
                elif s <= str_:
                    r_, u_, p_ = rr * (ps / pr) ** (1.0 / g), us, ps
                else:
                    c = 2.0 / gp * (cr - gm / 2.0 * (ur - s))
                    u_ = 2.0 / gp * (-cr + gm / 2.0 * ur + s)
                    r_ = rr * (c / cr) ** (2.0 / gm)
                    p_ = pr * (c / cr) ** (2.0 * g / gm)
        rho[n], u[n], p[n] = r_, u_, p_
    return rho, u, p


def vacuum_fan(xi, rl, pl, g):
    """Gas at rest (rho_L, p_L) expanding into vacuum on the right: (rho, u) at xi = (x-x0)/t.
    Head at xi = -c_L, front at xi = 2 c_L/(g-1)."""
    cl = math.sqrt(g * pl / rl)
    rho = np.zeros_like(xi)
    u = np.zeros_like(xi)
    head = xi <= -cl
    fan = (~head) & (xi < 2.0 * cl / (g - 1.0))
    rho[head] = rl
    base = 2.0 / (g + 1.0) - (g - 1.0) / (g + 1.0) * xi[fan] / cl
    rho[fan] = rl * base ** (2.0 / (g - 1.0))
    u[fan] = 2.0 / (g + 1.0) * (cl + xi[fan])
    return rho, u
