"""ctypes binding of the CPU oracle (oracle/csph_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
shares nothing with the CUDA path (paper_1912_04855_b200/csrc) and neither
imports the other.

The oracle states one CSPH-TVD time step (section 2.2, Eq. (4)-(8))
under the readings listed in DESIGN.md section 3.  This file only marshals
numpy arrays; all arithmetic is in the C++ file.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcsph_oracle.so")

F64, F32 = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_INFLOW = 0, 1, 2
LIMITER_MINMOD, LIMITER_VANLEER = 0, 1
RIEMANN_HLL, RIEMANN_LF, RIEMANN_HLLC = 0, 1, 2
KERNEL_CUBIC_SPLINE, KERNEL_POLY5 = 0, 1

_lib = None


def build(force=False):
    """Compile the oracle with gcc (oracle/build.sh).  Building is not using."""
    src = os.path.join(_HERE, "csph_oracle.cpp")
    if (not force and os.path.exists(_LIB_PATH)
            and os.path.getmtime(_LIB_PATH) >= os.path.getmtime(src)):
        return _LIB_PATH
    subprocess.check_call(["sh", os.path.join(_HERE, "build.sh")])
    return _LIB_PATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = ctypes.CDLL(_LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    lib.orc_set_threads.argtypes = [ci]
    lib.orc_set_threads.restype = None
    lib.orc_create.argtypes = [ci, ci, ci, cd, cd, ctypes.POINTER(ci), ci]
    lib.orc_create.restype = vp
    lib.orc_destroy.argtypes = [vp]
    lib.orc_destroy.restype = None
    lib.orc_set_state.argtypes = [vp] * 7
    lib.orc_set_state.restype = None
    lib.orc_compute_dt.argtypes = [vp, cd]
    lib.orc_compute_dt.restype = cd
    lib.orc_step.argtypes = [vp, cd]
    lib.orc_set_limiter.argtypes = [vp, ci]
    lib.orc_set_riemann.argtypes = [vp, ci]
    lib.orc_set_riemann.restype = None
    lib.orc_set_kernel.argtypes = [vp, ci]
    lib.orc_set_kernel.restype = None
    lib.orc_set_limiter.restype = None
    lib.orc_step.restype = None
    lib.orc_get_conserved.argtypes = [vp] * 6
    lib.orc_get_conserved.restype = None
    lib.orc_set_conserved.argtypes = [vp] * 6
    lib.orc_set_conserved.restype = None
    lib.orc_get_state.argtypes = [vp] * 6
    lib.orc_get_state.restype = None
    lib.orc_get_vacuum_mask.argtypes = [vp, vp]
    lib.orc_get_vacuum_mask.restype = None
    lib.orc_eval_force.argtypes = [vp] * 4
    lib.orc_eval_force.restype = None
    lib.orc_eval_Q.argtypes = [vp] * 8
    lib.orc_eval_Q.restype = None
    lib.orc_get_padded.argtypes = [vp, ci, vp]
    lib.orc_get_padded.restype = None
    lib.orc_get_offsets.argtypes = [vp, ci, ci, vp]
    lib.orc_get_offsets.restype = None
    lib.orc_lattice_constants.argtypes = [vp, ctypes.POINTER(cd)]
    lib.orc_lattice_constants.restype = None
    _lib = lib
    return lib


def set_threads(t):
    """Threads for the OpenMP split of each pass's outer (z) loop; results are
    bit-identical for any count (every cell is one and the same expression)."""
    _load().orc_set_threads(int(t))


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data)


class Oracle:
    """One grid.  Arrays are numpy, shape (nz, ny, nx) (x fastest), C order."""

    def __init__(self, nx, ny, nz, h, gamma, bc, dtype=F64):
        lib = _load()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.dtype = dtype
        self.np_dtype = np.float64 if dtype == F64 else np.float32
        bc_arr = (ctypes.c_int * 6)(*[int(b) for b in bc])
        self._h = lib.orc_create(self.nx, self.ny, self.nz, float(h), float(gamma), bc_arr, int(dtype))
        if not self._h:
            raise ValueError("orc_create rejected its arguments")

    def close(self):
        if getattr(self, "_h", None):
            _load().orc_destroy(self._h)
            self._h = None

    __del__ = close

    def _in(self, a):
        a = np.ascontiguousarray(a, dtype=self.np_dtype)
        assert a.shape == self.shape, (a.shape, self.shape)
        return a

    def _out(self, n):
        return [np.empty(self.shape, dtype=self.np_dtype) for _ in range(n)]

    def set_state(self, rho, u, v, w, p, psi):
        arrs = [self._in(a) for a in (rho, u, v, w, p, psi)]
        _load().orc_set_state(self._h, *[_ptr(a) for a in arrs])

    def compute_dt(self, cfl):
        return float(_load().orc_compute_dt(self._h, float(cfl)))

    def set_kernel(self, kernel):
        """0 = cubic spline (default, reading G5), 1 = W ~ (1 - q^2/4)^5 (no square root)."""
        _load().orc_set_kernel(self._h, int(kernel))

    def set_limiter(self, limiter):
        """0 = minmod (default, reading G12), 1 = van Leer."""
        _load().orc_set_limiter(self._h, int(limiter))

    def set_riemann(self, riemann):
        """0 = HLL (default, reading G13), 1 = local Lax-Friedrichs (G13b), 2 = HLLC (G13c)."""
        _load().orc_set_riemann(self._h, int(riemann))

    def step(self, dt):
        _load().orc_step(self._h, float(dt))

    def get_conserved(self):
        out = self._out(5)
        _load().orc_get_conserved(self._h, *[_ptr(a) for a in out])
        return out

    def set_conserved(self, rho, mx, my, mz, E):
        arrs = [self._in(a) for a in (rho, mx, my, mz, E)]
        _load().orc_set_conserved(self._h, *[_ptr(a) for a in arrs])

    def get_state(self):
        out = self._out(5)
        _load().orc_get_state(self._h, *[_ptr(a) for a in out])
        return out

    def get_vacuum_mask(self):
        m = np.empty(self.shape, dtype=np.uint8)
        _load().orc_get_vacuum_mask(self._h, _ptr(m))
        return m

    def eval_force(self):
        out = self._out(3)
        _load().orc_eval_force(self._h, *[_ptr(a) for a in out])
        return out

    def eval_Q(self, xi=None):
        """Q of Eq. (7) (momentum x3, energy) of the current state for particle
        offsets xi = (xi_x, xi_y, xi_z) or None (particles at the centres)."""
        out = self._out(4)
        if xi is None:
            xin = [ctypes.c_void_p(0)] * 3
        else:
            keep = [self._in(a) for a in xi]
            xin = [_ptr(a) for a in keep]
        _load().orc_eval_Q(self._h, *xin, *[_ptr(a) for a in out])
        return out

    def get_padded(self, c):
        """Component c of U^n with its 3 ghost layers per face as the next step's ghost fill leaves them,
        shape (nz+6, ny+6, nx+6)."""
        out = np.empty((self.nz + 6, self.ny + 6, self.nx + 6), dtype=self.np_dtype)
        _load().orc_get_padded(self._h, int(c), _ptr(out))
        return out

    def get_offsets(self, which, d):
        """Component d of the particle offsets of the last step, padded (nz+6, ny+6, nx+6): which = 0: xi* of
        Eq. (5), valid on interior(+)2; which = 1: xi^{n+1} of Eq. (6), valid on interior(+)1."""
        out = np.empty((self.nz + 6, self.ny + 6, self.nx + 6), dtype=self.np_dtype)
        _load().orc_get_offsets(self._h, int(which), int(d), _ptr(out))
        return out

    def lattice_constants(self):
        out = (ctypes.c_double * 4)()
        _load().orc_lattice_constants(self._h, out)
        return tuple(out)
