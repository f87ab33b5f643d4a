"""Thin Python binding of the C ABI in include/cspt.h (same names, argument marshalling
only).  PyTorch supplies device memory and streams; every step of the method runs in
the CUDA kernels of libcspt.so.  There is no CPU fallback: if the library is missing
or no CUDA device is present the calls fail loudly.
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcspt.so")

F64, F32 = 0, 1
BC_PERIODIC, BC_OUTFLOW, BC_INFLOW, BC_EXTERNAL = 0, 1, 2, 3
HALO_U, HALO_PSI = 0, 1
LIMITER_MINMOD, LIMITER_VANLEER = 0, 1
KERNEL_CUBIC_SPLINE, KERNEL_POLY5 = 0, 1
RIEMANN_HLL, RIEMANN_LF, RIEMANN_HLLC = 0, 1, 2
OK, EINVAL, ENOMEM, ECUDA, ESTATE, ELIMIT = 0, -1, -2, -3, -4, -5

# every symbol include/cspt.h declares: (name, restype, argtypes)
_vp, _ci, _cd, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
_pd = ctypes.POINTER(ctypes.c_double)
SYMBOLS = [
    ("cspt_workspace_bytes", _sz, [_ci, _ci, _ci, _ci]),
    ("cspt_create", _ci, [ctypes.POINTER(_vp), _ci, _ci, _ci, _cd, _cd, ctypes.POINTER(_ci), _ci, _vp, _sz, _vp]),
    ("cspt_set_state", _ci, [_vp] * 7),
    ("cspt_set_state_host", _ci, [_vp] * 7),
    ("cspt_set_state_host_async", _ci, [_vp] * 7),
    ("cspt_compute_dt", _ci, [_vp, _cd, _pd]),
    ("cspt_set_kernel", _ci, [_vp, _ci]),
    ("cspt_set_limiter", _ci, [_vp, _ci]),
    ("cspt_set_riemann", _ci, [_vp, _ci]),
    ("cspt_step", _ci, [_vp, _cd]),
    ("cspt_step_cfl", _ci, [_vp, _cd, _pd]),
    ("cspt_run_cfl", _ci, [_vp, _cd, _ci, _pd]),
    ("cspt_get_state", _ci, [_vp] * 6),
    ("cspt_get_conserved", _ci, [_vp] * 6),
    ("cspt_get_conserved_host", _ci, [_vp] * 6),
    ("cspt_get_conserved_host_async", _ci, [_vp] * 6),
    ("cspt_set_conserved", _ci, [_vp] * 6),
    ("cspt_get_vacuum_mask", _ci, [_vp, _vp]),
    ("cspt_launch_count", ctypes.c_longlong, [_vp]),
    ("cspt_profile_enable", _ci, [_vp, _ci]),
    ("cspt_profile_kernel_count", _ci, []),
    ("cspt_profile_kernel_name", ctypes.c_char_p, [_ci]),
    ("cspt_profile_read", _ci, [_vp, _ci, _pd, ctypes.POINTER(ctypes.c_longlong)]),
    ("cspt_probe_fma_rate", _ci, [_vp, _ci, _pd]),
    ("cspt_probe_fma_rate_ms", _ci, [_vp, _ci, _cd, _pd]),
    ("cspt_sm_count", _ci, [_vp]),
    ("cspt_debug_force_vacuum_variant", _ci, [_vp, _ci]),
    ("cspt_debug_tile_skip", _ci, [_vp, _ci]),
    ("cspt_debug_dead_ctas", _ci, [_vp, ctypes.POINTER(ctypes.c_longlong)]),
    ("cspt_halo_elems", _ci, [_vp, _ci, ctypes.POINTER(ctypes.c_longlong)]),
    ("cspt_halo_get", _ci, [_vp, _ci, _ci, _vp]),
    ("cspt_halo_put", _ci, [_vp, _ci, _ci, _vp]),
    ("cspt_finish_state", _ci, [_vp]),
    ("cspt_fill_ghosts", _ci, [_vp]),
    ("cspt_step_filled", _ci, [_vp, _cd]),
    ("cspt_smax_device", _ci, [_vp, ctypes.POINTER(_vp)]),
    ("cspt_step_filled_cfl", _ci, [_vp, _cd, _pd]),
    ("cspt_noalloc_max_cells", ctypes.c_longlong, []),
    ("cspt_cfl_dt_noalloc", _ci, [_ci, ctypes.c_longlong, _vp, _vp, _vp, _vp, _vp, _cd, _cd, _cd, _vp, _vp]),
    ("cspt_cuda_error", _ci, [_vp]),
    ("cspt_sync", _ci, [_vp]),
    ("cspt_destroy", None, [_vp]),
    ("cspt_strerror", ctypes.c_char_p, [_ci]),
]

_lib = None


class CsptError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().cspt_strerror(code).decode() if _lib is not None else str(code)
        super().__init__("%s: %s (%d)" % (where, msg, code))


def lib():
    """Loads libcspt.so (built by `python -m paper_1912_04855_b200.build`); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libcspt.so is missing: run `python -m paper_1912_04855_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        for name, res, args in SYMBOLS:
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(code, where):
    if code != OK:
        raise CsptError(code, where)


def _dptr(t):
    return ctypes.c_void_p(t.data_ptr())


def noalloc_max_cells():
    """Largest ncells cspt_cfl_dt_noalloc accepts (its scratch is a fixed array inside the library)."""
    return int(lib().cspt_noalloc_max_cells())


def cfl_dt_noalloc(rho, mx, my, mz, E, gamma, h, cfl, out, stream=None):
    """cspt_cfl_dt_noalloc: the CFL time step of five dense, contiguous CUDA tensors of conserved variables, written
    into the caller's one-element CUDA tensor `out` of the same dtype (float64 or float32).  For callers that hold the
    fields but cannot allocate a ctx workspace (all memory in the application's own pool, no cudaMalloc allowed in the
    time loop, plug-in monitors that only receive pointers): neither this binding nor the library allocates anything,
    which is why `out` is an argument and not a return value.  Enqueues on `stream` (default: torch's current stream)
    and does not sync; calls on one device must not overlap (they share the library's built-in scratch).  Sizes
    above noalloc_max_cells() raise CsptError with code ELIMIT."""
    import torch
    ts = (rho, mx, my, mz, E)
    dt = ts[0].dtype
    assert dt in (torch.float64, torch.float32)
    assert all(t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() == ts[0].numel() for t in ts)
    assert out.is_cuda and out.dtype == dt and out.numel() == 1 and out.device == ts[0].device
    assert torch.cuda.current_device() == ts[0].device.index, "make the tensors' device current first"
    st = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().cspt_cfl_dt_noalloc(F64 if dt == torch.float64 else F32, ts[0].numel(), *[_dptr(t) for t in ts],
                                     float(gamma), float(h), float(cfl), _dptr(out), ctypes.c_void_p(st.cuda_stream)),
           "cspt_cfl_dt_noalloc")
    return out


class Solver:
    """One grid on the current CUDA device.  Tensors are (nz, ny, nx), x fastest."""

    def __init__(self, nx, ny, nz, h, gamma, bc, dtype=F64, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("cspt needs a CUDA device (there is no CPU fallback)")
        L = lib()
        self.torch = torch
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.dtype = dtype
        self.tdtype = torch.float64 if dtype == F64 else torch.float32
        self.device = torch.device("cuda", torch.cuda.current_device())
        nbytes = L.cspt_workspace_bytes(self.nx, self.ny, self.nz, int(dtype))
        if nbytes == 0:
            raise CsptError(EINVAL, "cspt_workspace_bytes")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        h_ = ctypes.c_void_p()
        bc_arr = (ctypes.c_int * 6)(*[int(b) for b in bc])
        _check(L.cspt_create(ctypes.byref(h_), self.nx, self.ny, self.nz, float(h), float(gamma), bc_arr, int(dtype),
                             ctypes.c_void_p(self.workspace.data_ptr()), nbytes,
                             ctypes.c_void_p(self.stream.cuda_stream)), "cspt_create")
        self._h = h_

    def close(self):
        if getattr(self, "_h", None):
            self.torch.cuda.synchronize()
            lib().cspt_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers ---------------------------------------------------------------------
    def _dev(self, a):
        t = self.torch.as_tensor(a)
        t = t.to(device=self.device, dtype=self.tdtype).contiguous()
        assert tuple(t.shape) == self.shape, (tuple(t.shape), self.shape)
        return t

    def _host(self, a):
        t = self.torch.as_tensor(a)
        assert t.device.type == "cpu" and t.dtype == self.tdtype and t.is_contiguous() and tuple(t.shape) == self.shape
        return t

    def _empty(self, n, dtype=None):
        return [self.torch.empty(self.shape, dtype=dtype or self.tdtype, device=self.device) for _ in range(n)]

    # stream hand-over: tensors arrive from / go to torch's current stream, the library works on self.stream
    def _before(self):
        self.stream.wait_stream(self.torch.cuda.current_stream())

    def _after(self):
        self.torch.cuda.current_stream().wait_stream(self.stream)

    # -- the C ABI, same names -----------------------------------------------------------
    def set_state(self, rho, u, v, w, p, psi):
        ts = [self._dev(a) for a in (rho, u, v, w, p, psi)]
        self._before()
        _check(lib().cspt_set_state(self._h, *[_dptr(t) for t in ts]), "cspt_set_state")
        self.stream.synchronize()      # inputs may be temporaries

    def set_state_host(self, rho, u, v, w, p, psi):
        ts = [self._host(a) for a in (rho, u, v, w, p, psi)]
        _check(lib().cspt_set_state_host(self._h, *[_dptr(t) for t in ts]), "cspt_set_state_host")

    def set_state_host_async(self, rho, u, v, w, p, psi):
        """Enqueues only: the (pinned) host tensors must stay untouched until sync()."""
        ts = [self._host(a) for a in (rho, u, v, w, p, psi)]
        _check(lib().cspt_set_state_host_async(self._h, *[_dptr(t) for t in ts]), "cspt_set_state_host_async")

    def compute_dt(self, cfl):
        out = ctypes.c_double()
        _check(lib().cspt_compute_dt(self._h, float(cfl), ctypes.byref(out)), "cspt_compute_dt")
        return out.value

    def set_kernel(self, kernel):
        _check(lib().cspt_set_kernel(self._h, int(kernel)), "cspt_set_kernel")

    def set_limiter(self, limiter):
        _check(lib().cspt_set_limiter(self._h, int(limiter)), "cspt_set_limiter")

    def set_riemann(self, riemann):
        _check(lib().cspt_set_riemann(self._h, int(riemann)), "cspt_set_riemann")

    def step(self, dt):
        _check(lib().cspt_step(self._h, float(dt)), "cspt_step")

    def step_cfl(self, cfl, want_dt=False):
        if want_dt:
            out = ctypes.c_double()
            _check(lib().cspt_step_cfl(self._h, float(cfl), ctypes.byref(out)), "cspt_step_cfl")
            return out.value
        _check(lib().cspt_step_cfl(self._h, float(cfl), None), "cspt_step_cfl")
        return None

    def run_cfl(self, cfl, nsteps, want_time=False):
        """nsteps CFL-limited steps from a CUDA graph; returns the time since set_state if want_time."""
        if want_time:
            out = ctypes.c_double()
            _check(lib().cspt_run_cfl(self._h, float(cfl), int(nsteps), ctypes.byref(out)), "cspt_run_cfl")
            return out.value
        _check(lib().cspt_run_cfl(self._h, float(cfl), int(nsteps), None), "cspt_run_cfl")
        return None

    def get_state(self):
        out = self._empty(5)
        self._before()
        _check(lib().cspt_get_state(self._h, *[_dptr(t) for t in out]), "cspt_get_state")
        self._after()
        return out

    def get_conserved(self):
        out = self._empty(5)
        self._before()
        _check(lib().cspt_get_conserved(self._h, *[_dptr(t) for t in out]), "cspt_get_conserved")
        self._after()
        return out

    def get_conserved_host(self, out):
        ts = [self._host(a) for a in out]
        _check(lib().cspt_get_conserved_host(self._h, *[_dptr(t) for t in ts]), "cspt_get_conserved_host")
        return out

    def get_conserved_host_async(self, out):
        """Enqueues only: `out` holds the result after sync()."""
        ts = [self._host(a) for a in out]
        _check(lib().cspt_get_conserved_host_async(self._h, *[_dptr(t) for t in ts]), "cspt_get_conserved_host_async")
        return out

    def set_conserved(self, rho, mx, my, mz, E):
        ts = [self._dev(a) for a in (rho, mx, my, mz, E)]
        self._before()
        _check(lib().cspt_set_conserved(self._h, *[_dptr(t) for t in ts]), "cspt_set_conserved")
        self.stream.synchronize()

    def get_vacuum_mask(self):
        m = self.torch.empty(self.shape, dtype=self.torch.uint8, device=self.device)
        self._before()
        _check(lib().cspt_get_vacuum_mask(self._h, _dptr(m)), "cspt_get_vacuum_mask")
        self._after()
        return m

    def launch_count(self):
        return int(lib().cspt_launch_count(self._h))

    def profile_enable(self, on=True):
        _check(lib().cspt_profile_enable(self._h, 1 if on else 0), "cspt_profile_enable")

    def profile_read(self):
        """{kernel name: (total device ms, launches)} since profile_enable(True)."""
        L = lib()
        out = {}
        for kid in range(L.cspt_profile_kernel_count()):
            ms, n = ctypes.c_double(), ctypes.c_longlong()
            _check(L.cspt_profile_read(self._h, kid, ctypes.byref(ms), ctypes.byref(n)), "cspt_profile_read")
            if n.value:
                out[L.cspt_profile_kernel_name(kid).decode()] = (ms.value, int(n.value))
        return out

    def probe_fma_rate(self, other_per_fma=0, min_ms=0.0):
        """Measured FMA rate of the plain FP pipe in the solver's precision (thread-level FMAs per second), alone or
        with 2 / 4 / 8 independent integer instructions interleaved per FMA; min_ms > 0 repeats the probe until it has
        run that long (cspt_probe_fma_rate_ms)."""
        out = ctypes.c_double()
        if min_ms:
            _check(lib().cspt_probe_fma_rate_ms(self._h, int(other_per_fma), float(min_ms), ctypes.byref(out)),
                   "cspt_probe_fma_rate_ms")
        else:
            _check(lib().cspt_probe_fma_rate(self._h, int(other_per_fma), ctypes.byref(out)), "cspt_probe_fma_rate")
        return out.value

    def debug_tile_skip(self, on):
        _check(lib().cspt_debug_tile_skip(self._h, 1 if on else 0), "cspt_debug_tile_skip")

    def debug_dead_ctas(self):
        n = ctypes.c_longlong()
        _check(lib().cspt_debug_dead_ctas(self._h, ctypes.byref(n)), "cspt_debug_dead_ctas")
        return int(n.value)

    def debug_force_vacuum_variant(self, force):
        _check(lib().cspt_debug_force_vacuum_variant(self._h, int(force)), "cspt_debug_force_vacuum_variant")

    def sm_count(self):
        return int(lib().cspt_sm_count(self._h))

    # -- z-slab decomposition (include/cspt.h: CSPT_BC_EXTERNAL) ---------------------------------------
    def halo_elems(self, what=HALO_U):
        n = ctypes.c_longlong()
        _check(lib().cspt_halo_elems(self._h, int(what), ctypes.byref(n)), "cspt_halo_elems")
        return int(n.value)

    def halo_get(self, face, what=HALO_U, out=None):
        if out is None:
            out = self.torch.empty(self.halo_elems(what), dtype=self.tdtype, device=self.device)
        self._before()
        _check(lib().cspt_halo_get(self._h, int(face), int(what), _dptr(out)), "cspt_halo_get")
        self._after()
        return out

    def halo_put(self, face, buf, what=HALO_U):
        assert buf.is_cuda and buf.dtype == self.tdtype and buf.is_contiguous() and buf.numel() == self.halo_elems(what)
        self._before()
        _check(lib().cspt_halo_put(self._h, int(face), int(what), _dptr(buf)), "cspt_halo_put")
        self._after()

    def finish_state(self):
        _check(lib().cspt_finish_state(self._h), "cspt_finish_state")

    def fill_ghosts(self):
        _check(lib().cspt_fill_ghosts(self._h), "cspt_fill_ghosts")

    def step_filled(self, dt):
        _check(lib().cspt_step_filled(self._h, float(dt)), "cspt_step_filled")

    def smax_device(self):
        """The slab's maximum signal speed as a one-element tensor VIEW of the word in the workspace (no copy): reduce
        it in place over the slabs (all_reduce MAX on the solver's stream), then step_filled_cfl."""
        p = ctypes.c_void_p()
        self._before()
        _check(lib().cspt_smax_device(self._h, ctypes.byref(p)), "cspt_smax_device")
        self._after()
        off = p.value - self.workspace.data_ptr()
        esz = 8 if self.dtype == F64 else 4
        assert 0 <= off and off + esz <= self.workspace.numel() and off % esz == 0
        return self.workspace[off:off + esz].view(self.tdtype)

    def step_filled_cfl(self, cfl, want_dt=False):
        self._before()
        if want_dt:
            out = ctypes.c_double()
            _check(lib().cspt_step_filled_cfl(self._h, float(cfl), ctypes.byref(out)), "cspt_step_filled_cfl")
            return out.value
        _check(lib().cspt_step_filled_cfl(self._h, float(cfl), None), "cspt_step_filled_cfl")
        return None

    def cuda_error(self):
        return int(lib().cspt_cuda_error(self._h))

    def sync(self):
        _check(lib().cspt_sync(self._h), "cspt_sync")
