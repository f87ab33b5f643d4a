"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench,
so it holds none of the method's arithmetic: it only evaluates the initial
primitive fields (rho, u, v, w, p) and the potential psi at cell centres.  It
imports neither `oracle/` nor the CUDA binding.  numpy only.

Every field is a pure function of the GLOBAL integer cell index, so any window
of any config can be regenerated from coordinates alone (used by the full-size
windowed parity tests).  Random numbers come from a counter-based generator
(splitmix64 of seed*2^32 + linear cell index), never from a stateful stream.

Arrays have shape (nz, ny, nx), x fastest.
"""
import math

import numpy as np

PERIODIC, OUTFLOW, INFLOW = 0, 1, 2

_M64 = (1 << 64) - 1


def splitmix64(x):
    """Counter-based generator: numpy uint64 array -> uint64 array."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed, counter):
    """Uniform [0,1) doubles from (seed, counter array)."""
    with np.errstate(over="ignore"):
        key = np.uint64((int(seed) << 32) & _M64) + np.asarray(counter, dtype=np.uint64)
    return (splitmix64(key) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


class Workload:
    """Description of one config at grid size (nx, ny, nz)."""

    def __init__(self, name, nx, ny, nz, h, gamma, bc, origin, cfl, steps, dtype, fields, t_end=None):
        self.name = name
        self.nx, self.ny, self.nz = nx, ny, nz
        self.h, self.gamma = h, gamma
        self.bc = tuple(bc)                # xlo,xhi,ylo,yhi,zlo,zhi
        self.origin = origin               # coordinate of the low corner of cell (0,0,0)
        self.cfl, self.steps, self.t_end = cfl, steps, t_end
        self.dtype = dtype                 # "f64" | "f32"
        self._fields = fields              # fn(ix, iy, iz) -> 6 float64 arrays

    @property
    def cells(self):
        return self.nx * self.ny * self.nz

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32

    def wrap(self, idx, axis):
        """Map global indices outside the grid onto it the way the axis's boundary does
        for the INITIAL data (periodic wrap; otherwise the analytic field is simply
        evaluated where it is asked for - callers clip windows at non-periodic faces)."""
        n = (self.nx, self.ny, self.nz)[axis]
        if self.bc[2 * axis] == PERIODIC:
            return np.mod(idx, n)
        return idx

    def fields(self, ix=None, iy=None, iz=None):
        """(rho,u,v,w,p,psi) on the index box ix x iy x iz (1-D int arrays of GLOBAL cell
        indices; default: the whole grid), cast to the workload dtype."""
        ix = np.arange(self.nx) if ix is None else np.asarray(ix)
        iy = np.arange(self.ny) if iy is None else np.asarray(iy)
        iz = np.arange(self.nz) if iz is None else np.asarray(iz)
        ix, iy, iz = self.wrap(ix, 0), self.wrap(iy, 1), self.wrap(iz, 2)
        out = self._fields(ix.astype(np.int64), iy.astype(np.int64), iz.astype(np.int64))
        shape = (len(iz), len(iy), len(ix))
        return tuple(np.ascontiguousarray(np.broadcast_to(a, shape), dtype=self.np_dtype) for a in out)

    def fields_slab(self, k0, k1):
        """Whole-xy slab k0 <= k < k1 (for filling large grids piecewise)."""
        return self.fields(iz=np.arange(k0, k1))


def _centres(idx, origin, h):
    return origin + (idx.astype(np.float64) + 0.5) * h


def _b(ax, arr):
    """1-D array along axis ax in {0:x,1:y,2:z} -> broadcastable (nz,ny,nx) view."""
    shp = [1, 1, 1]
    shp[2 - ax] = len(arr)
    return arr.reshape(shp)


# ---- cfg1: Sod shock tube (BASELINE.json configs[0]) -------------------------
def sod(n=64, nt=4, axis=0, dtype="f64"):
    dims = [nt, nt, nt]
    dims[axis] = n
    h = 1.0 / n
    bc = [PERIODIC] * 6
    bc[2 * axis] = bc[2 * axis + 1] = OUTFLOW

    def f(ix, iy, iz):
        ia = (ix, iy, iz)[axis]
        left = _b(axis, (ia < n // 2).astype(np.float64))
        one = np.ones((1, 1, 1))
        rho = left * 1.0 + (1 - left) * 0.125
        p = left * 1.0 + (1 - left) * 0.1
        z = 0.0 * one
        return rho, z, z, z, p, z

    return Workload("sod", dims[0], dims[1], dims[2], h, 1.4, bc, (0.0, 0.0, 0.0), 0.4, None, dtype, f, t_end=0.2)


# ---- cfg2: Sedov-type point blast (configs[1]) -------------------------------
def sedov(n=128, dtype="f64"):
    h = 1.0 / n
    gamma = 1.4

    def f(ix, iy, iz):
        # distance (in cells) from the cell centre to the domain centre, a cell corner
        dx = _b(0, ix.astype(np.float64) + 0.5 - n / 2)
        dy = _b(1, iy.astype(np.float64) + 0.5 - n / 2)
        dz = _b(2, iz.astype(np.float64) + 0.5 - n / 2)
        hot = ((dx * dx + dy * dy) + dz * dz) < 4.0          # 32 cells
        p_hot = (gamma - 1.0) * 1.0 / (32.0 * h ** 3)       # E = 1 spread as pressure
        p = np.where(hot, p_hot, 1e-5)
        one = np.ones((1, 1, 1))
        z = 0.0 * one
        return one, z, z, z, p, z

    return Workload("sedov", n, n, n, h, gamma, [OUTFLOW] * 6, (0.0, 0.0, 0.0), 0.4, 200, dtype, f)


# ---- cfg3: supersonic flow through a Gaussian potential well (configs[2]) ----
def well(n=256, dtype="f64", variant="flow"):
    """variant: 'flow' (Mach 2 inflow), 'gamma2' (exact discrete equilibrium, all
    periodic), 'isothermal' (rho = p = exp(-psi), O(h^2) equilibrium)."""
    h = 1.0 / n
    gamma = 5.0 / 3.0
    a = 0.1
    org = (-0.5, -0.5, -0.5)
    if variant == "flow":
        bc = [INFLOW, OUTFLOW, PERIODIC, PERIODIC, PERIODIC, PERIODIC]
    else:
        bc = [PERIODIC] * 6

    def f(ix, iy, iz):
        x = _b(0, _centres(ix, org[0], h))
        y = _b(1, _centres(iy, org[1], h))
        z = _b(2, _centres(iz, org[2], h))
        psi = -np.exp(-((x * x + y * y) + z * z) / (a * a))
        one = np.ones((1, 1, 1))
        zero = 0.0 * one
        if variant == "flow":
            return one, 2.0 * math.sqrt(gamma) * one, zero, zero, one, psi
        if variant == "gamma2":
            phi = math.sqrt(2.0) - 0.8 * psi
            return 0.8 * phi, zero, zero, zero, 0.5 * phi * phi, psi
        if variant == "isothermal":
            r = np.exp(-psi)
            return r, zero, zero, zero, r, psi
        raise ValueError(variant)

    return Workload("well-" + variant, n, n, n, h, gamma, bc, org, 0.4, 100, dtype, f)


# ---- cfg4: smooth random periodic field (configs[3]) -------------------------
def turbulence(n=512, dtype="f64", seed=4):
    h = 2.0 * math.pi / n
    # phases[field, mode, axis], uniform [0, 2 pi)
    ph = 2.0 * math.pi * uniform01(seed, np.arange(4 * 8 * 3)).reshape(4, 8, 3)

    def f(ix, iy, iz):
        x = _centres(ix, 0.0, h)
        y = _centres(iy, 0.0, h)
        z = _centres(iz, 0.0, h)
        out = []
        for fld in range(4):
            acc = 0.0
            for k in range(1, 9):
                sx = _b(0, np.sin(k * x + ph[fld, k - 1, 0]))
                sy = _b(1, np.sin(k * y + ph[fld, k - 1, 1]))
                sz = _b(2, np.sin(k * z + ph[fld, k - 1, 2]))
                acc = acc + (sz * sy) * sx
            out.append(0.1 * acc)
        one = np.ones((1, 1, 1))
        return 1.0 + out[0], out[1], out[2], out[3], one, 0.0 * one

    return Workload("turbulence", n, n, n, h, 1.4, [PERIODIC] * 6, (0.0, 0.0, 0.0), 0.4, 50, dtype, f)


# ---- cfg5: rotating disk with a gas-vacuum boundary (configs[4]) -------------
def disk(n=1024, dtype="f32", seed=5):
    h = 1.0 / n
    gamma = 5.0 / 3.0
    b, Rd, hz, Rmax = 0.05, 0.1, 0.02, 0.4
    org = (-0.5, -0.5, -0.5)

    def f(ix, iy, iz):
        x = _b(0, _centres(ix, org[0], h))
        y = _b(1, _centres(iy, org[1], h))
        z = _b(2, _centres(iz, org[2], h))
        R2 = x * x + y * y
        R = np.sqrt(R2)
        s2 = R2 + z * z + b * b
        psi = -1.0 / np.sqrt(s2)
        lin = (_b(2, iz) * n + _b(1, iy)) * n + _b(0, ix)
        noise = 1.0 + 0.01 * (2.0 * uniform01(seed, lin) - 1.0)
        rho = np.where(R < Rmax, np.exp(-R / Rd) * np.exp(-(z * z) / (2.0 * hz * hz)) * noise, 0.0)
        vphi = np.sqrt(R2 / s2 ** 1.5)
        with np.errstate(invalid="ignore", divide="ignore"):
            cs = np.where(R > 0, x / R, 0.0)
            sn = np.where(R > 0, y / R, 0.0)
        gas = rho > 0
        u = np.where(gas, -vphi * sn, 0.0)
        v = np.where(gas, vphi * cs, 0.0)
        p = 0.01 * rho ** gamma
        return rho, u, v, 0.0 * rho, p, psi + 0.0 * rho

    return Workload("disk", n, n, n, h, gamma, [OUTFLOW] * 6, org, 0.4, 20, dtype, f)


# ---- a generic smooth random periodic state for parity tests ----------------
def random_smooth(nx, ny, nz, dtype="f64", seed=11, bc=None, gamma=1.4, with_psi=True):
    """Few-mode smooth fields with O(1) gradients on an arbitrary (ragged) grid;
    used by the element-by-element parity tests (not one of BASELINE's configs)."""
    h = 1.0 / max(nx, ny, nz)
    bc = [PERIODIC] * 6 if bc is None else list(bc)
    ph = 2.0 * math.pi * uniform01(seed, np.arange(6 * 3 * 3)).reshape(6, 3, 3)
    L = (nx * h, ny * h, nz * h)

    def f(ix, iy, iz):
        c = (_centres(ix, 0.0, h), _centres(iy, 0.0, h), _centres(iz, 0.0, h))
        out = []
        for fld in range(6):
            acc = 0.0
            for k in range(1, 4):
                s = [_b(ax, np.sin(2.0 * math.pi * k * c[ax] / L[ax] + ph[fld, k - 1, ax])) for ax in range(3)]
                acc = acc + (s[2] * s[1]) * s[0] / k
            out.append(acc)
        rho = 1.0 + 0.3 * out[0]
        p = 1.0 + 0.3 * out[4]
        psi = 0.2 * out[5] if with_psi else 0.0 * out[5]
        return rho, 0.5 * out[1], 0.5 * out[2], 0.5 * out[3], p, psi

    return Workload("random-smooth", nx, ny, nz, h, gamma, bc, (0.0, 0.0, 0.0), 0.4, 10, dtype, f)


def by_name(name, n=None, dtype=None):
    """The five BASELINE.json configs by short name, at full size unless n is given."""
    table = {
        "sod": (sod, 64, "f64"),
        "sedov": (sedov, 128, "f64"),
        "well": (well, 256, "f64"),
        "turbulence": (turbulence, 512, "f64"),
        "disk": (disk, 1024, "f32"),
    }
    fn, n0, d0 = table[name]
    return fn(n=n or n0, dtype=dtype or d0)
