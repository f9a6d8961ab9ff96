"""Thin ctypes binding of libgpupegas.so (include/gpupegas.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch appears here only to own
the device memory (one uint8 tensor bound with gp_bind_storage) and the CUDA stream.  If the
library is missing or no CUDA device is present the calls fail loudly; there is no fallback.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgpupegas.so")

GP_OK, GP_ERR_ARG, GP_ERR_ALLOC, GP_ERR_CUDA, GP_ERR_CUFFT, GP_ERR_STATE, GP_ERR_UNSUPPORTED = range(7)
GP_GAS, GP_STARS, GP_OD = 1, 2, 4
GP_POISSON_NONE, GP_POISSON_PERIODIC, GP_POISSON_ISOLATED = 0, 1, 2
GP_BC_PERIODIC, GP_BC_OUTFLOW = 0, 1
FIELDS = ["rho", "mx", "my", "mz", "E",
          "n", "nux", "nuy", "nuz", "Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz", "phi"]
# carried fields of the overdetermined system (GP_OD contexts): GP_EPS, GP_PXX ... GP_PZZ
OD_GAS_FIELDS, OD_STAR_FIELDS = ["eps"], ["Pxx", "Pxy", "Pxz", "Pyy", "Pyz", "Pzz"]
FIELD_ID = {name: i for i, name in enumerate(FIELDS + OD_GAS_FIELDS + OD_STAR_FIELDS)}
GAS_FIELDS, STAR_FIELDS = FIELDS[:5], FIELDS[5:15]

# the symbols include/gpupegas.h declares
EXPORTS = ["gp_create", "gp_destroy", "gp_set_state", "gp_get_state", "gp_solve_poisson", "gp_max_dt",
           "gp_step", "gp_last_error", "gp_set_stream", "gp_storage_bytes", "gp_bind_storage",
           "gp_synchronize", "gp_launch_counts", "gp_timing_enable", "gp_timing_read", "gp_math_selftest",
           "gp_fp64_rate_selftest", "gp_od_derive", "gp_od_step", "gp_od_balance", "gp_kappa", "gp_od_last_kappa",
           "gp_kappa_noalloc"]
KAPPA_NOALLOC_MAX_CELLS = 134217728      # GP_KAPPA_NOALLOC_MAX_CELLS


class gp_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("h", C.c_double),
                ("components", C.c_int), ("poisson", C.c_int), ("G", C.c_double)]


class gp_bc(C.Structure):
    _fields_ = [("x", C.c_int), ("y", C.c_int), ("z", C.c_int)]


class GpError(RuntimeError):
    def __init__(self, code, what, text):
        super().__init__(f"{what}: error {code}: {text}")
        self.code = code


_lib = None


def lib():
    """Load libgpupegas.so (built in-tree by `python -m paper_1311_0861_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1311_0861_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        L.gp_create.restype = vp
        L.gp_create.argtypes = [C.POINTER(gp_grid), C.c_double, C.POINTER(gp_bc)]
        L.gp_destroy.restype = None
        L.gp_destroy.argtypes = [vp]
        L.gp_set_state.argtypes = [vp, C.c_int, vp, C.c_int]
        L.gp_get_state.argtypes = [vp, C.c_int, vp, C.c_int]
        L.gp_solve_poisson.argtypes = [vp]
        L.gp_max_dt.argtypes = [vp, C.c_double, dp]
        L.gp_step.argtypes = [vp, C.c_double]
        L.gp_last_error.restype = C.c_char_p
        L.gp_set_stream.argtypes = [vp, vp]
        L.gp_storage_bytes.restype = C.c_size_t
        L.gp_storage_bytes.argtypes = [C.POINTER(gp_grid)]
        L.gp_bind_storage.argtypes = [vp, vp, C.c_size_t]
        L.gp_synchronize.argtypes = [vp]
        L.gp_launch_counts.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.gp_timing_enable.argtypes = [vp, C.c_int]
        L.gp_timing_read.argtypes = [vp, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_char_p), dp, C.POINTER(C.c_longlong)]
        L.gp_math_selftest.argtypes = [C.c_int, vp, vp, vp]
        L.gp_fp64_rate_selftest.argtypes = [dp, dp]
        L.gp_od_derive.argtypes = [vp]
        L.gp_od_step.argtypes = [vp, C.c_double, C.c_int]
        L.gp_od_balance.argtypes = [vp]
        L.gp_kappa.argtypes = [vp, dp]
        L.gp_od_last_kappa.argtypes = [vp, dp]
        L.gp_kappa_noalloc.argtypes = [C.c_size_t, C.c_double, vp, vp, vp, vp]
        _lib = L
    return _lib


def math_selftest(x):
    """(1/x, 1/sqrt(x)) as the hydro kernels compute them, for a numpy float64 array x > 0."""
    import numpy as np
    x = np.ascontiguousarray(x, dtype=np.float64).ravel()
    r, s = np.empty_like(x), np.empty_like(x)
    _chk(lib().gp_math_selftest(x.size, x.ctypes.data, r.ctypes.data, s.ctypes.data), "gp_math_selftest")
    return r, s


def fp64_rate_selftest():
    """(fp64 thread-instructions per second, kernel ms) of the DFMA self test on the current device."""
    rate, ms = C.c_double(0.0), C.c_double(0.0)
    _chk(lib().gp_fp64_rate_selftest(C.byref(rate), C.byref(ms)), "gp_fp64_rate_selftest")
    return rate.value, ms.value


def kappa_noalloc(h, gas=None, stars=None, out=None, stream=None):
    """gp_kappa_noalloc: (kappa_gas, kappa_bme) of fields the caller already holds on the device, for programs that
    cannot let the library allocate (all HBM already spoken for by the caller's own pool, or a loop that must not
    stall on cudaMalloc).  `gas`: 6 float64 CUDA tensors (rho, mx, my, mz, E, eps), `stars`: 16 (n, nu*, E**, P**),
    all of the same number of elements, contiguous; `out`: a float64 CUDA tensor of 2 elements (the caller's too:
    nothing is allocated here), returned.  Asynchronous on `stream` (default: torch's current stream).  The
    library's one fixed scratch array is shared by all calls on a GPU, so do not let two calls overlap."""
    import torch
    groups = [g for g in (gas, stars) if g is not None]
    assert groups and out is not None and out.is_cuda and out.dtype == torch.float64 and out.numel() == 2
    assert (gas is None or len(gas) == 6) and (stars is None or len(stars) == 16)
    n = groups[0][0].numel()
    for g in groups:
        for t in g:
            assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n
    as_ptrs = lambda g: None if g is None else (C.c_void_p * len(g))(*[t.data_ptr() for t in g])
    st = stream if stream is not None else torch.cuda.current_stream()
    _chk(lib().gp_kappa_noalloc(n, h, as_ptrs(gas), as_ptrs(stars), out.data_ptr(), st.cuda_stream), "gp_kappa_noalloc")
    return out


def _chk(code, what):
    if code != GP_OK:
        raise GpError(code, what, lib().gp_last_error().decode())


class Simulation:
    """One grid + state on the current CUDA device.  Host arrays are numpy float64 (nz, ny, nx)."""

    def __init__(self, nx, ny, nz, h, components=GP_GAS, poisson=GP_POISSON_NONE, G=1.0, gamma=5.0 / 3.0,
                 bc=(GP_BC_PERIODIC,) * 3, use_torch_memory=True, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1311_0861_b200 needs a CUDA device; there is no CPU path")
        L = lib()
        self.nx, self.ny, self.nz, self.h = nx, ny, nz, h
        self.shape = (nz, ny, nx)
        self.cells = nx * ny * nz
        self.components, self.poisson = components, poisson
        self._grid = gp_grid(nx, ny, nz, h, components, poisson, G)
        self._bc = gp_bc(*bc)
        self._c = L.gp_create(C.byref(self._grid), gamma, C.byref(self._bc))
        if not self._c:
            raise GpError(GP_ERR_ARG, "gp_create", L.gp_last_error().decode())
        self._storage = None
        if use_torch_memory:
            nbytes = L.gp_storage_bytes(C.byref(self._grid))
            self._storage = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            ptr = (self._storage.data_ptr() + 255) & ~255
            _chk(L.gp_bind_storage(self._c, ptr, nbytes), "gp_bind_storage")
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        _chk(L.gp_set_stream(self._c, self._stream.cuda_stream), "gp_set_stream")

    @classmethod
    def from_workload(cls, w, **kw):
        return cls(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc, **kw)

    def close(self):
        if getattr(self, "_c", None):
            lib().gp_destroy(self._c)
            self._c = None
            self._storage = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def field_names(self):
        return (GAS_FIELDS if self.components & GP_GAS else []) + (STAR_FIELDS if self.components & GP_STARS else [])

    def od_field_names(self):
        """The carried fields of a GP_OD context."""
        if not self.components & GP_OD:
            return []
        return (OD_GAS_FIELDS if self.components & GP_GAS else []) + (OD_STAR_FIELDS if self.components & GP_STARS else [])

    # ---- state in / out -------------------------------------------------------------------
    def set(self, name, arr):
        """arr: numpy float64 array (host) or a torch float64 CUDA tensor of nz*ny*nx elements."""
        import numpy as np
        import torch
        if isinstance(arr, torch.Tensor):
            assert arr.is_cuda and arr.dtype == torch.float64 and arr.is_contiguous() and arr.numel() == self.cells
            _chk(lib().gp_set_state(self._c, FIELD_ID[name], arr.data_ptr(), 1), f"gp_set_state({name})")
        else:
            a = np.ascontiguousarray(arr, dtype=np.float64)
            assert a.size == self.cells, (a.shape, self.shape)
            _chk(lib().gp_set_state(self._c, FIELD_ID[name], a.ctypes.data, 0), f"gp_set_state({name})")

    def set_state(self, state):
        for k, v in state.items():
            self.set(k, v)

    def get(self, name, out=None):
        import numpy as np
        import torch
        if isinstance(out, torch.Tensor):
            assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.cells
            _chk(lib().gp_get_state(self._c, FIELD_ID[name], out.data_ptr(), 1), f"gp_get_state({name})")
            return out
        if out is None:
            out = np.empty(self.shape, dtype=np.float64)
        assert out.flags.c_contiguous and out.dtype == np.float64 and out.size == self.cells
        _chk(lib().gp_get_state(self._c, FIELD_ID[name], out.ctypes.data, 0), f"gp_get_state({name})")
        return out

    def get_state(self):
        return {k: self.get(k) for k in self.field_names()}

    # ---- the hot path ---------------------------------------------------------------------
    def solve_poisson(self):
        _chk(lib().gp_solve_poisson(self._c), "gp_solve_poisson")

    def max_dt(self, cfl, to_host=True):
        if not to_host:
            _chk(lib().gp_max_dt(self._c, cfl, None), "gp_max_dt")
            return None
        dt = C.c_double(0.0)
        _chk(lib().gp_max_dt(self._c, cfl, C.byref(dt)), "gp_max_dt")
        return dt.value

    def step(self, dt=0.0):
        """dt > 0: use it; dt <= 0: use the device-resident dt of the last max_dt."""
        _chk(lib().gp_step(self._c, dt), "gp_step")

    # ---- overdetermined system (GP_OD contexts) -------------------------------------------
    def od_derive(self):
        _chk(lib().gp_od_derive(self._c), "gp_od_derive")

    def od_step(self, dt=0.0, balance=True):
        _chk(lib().gp_od_step(self._c, dt, 1 if balance else 0), "gp_od_step")

    def od_balance(self):
        _chk(lib().gp_od_balance(self._c), "gp_od_balance")

    def kappa(self):
        """(kappa_gas, kappa_bme) of the current state."""
        out = (C.c_double * 2)()
        _chk(lib().gp_kappa(self._c, out), "gp_kappa")
        return out[0], out[1]

    def od_last_kappa(self):
        """(kappa_gas, kappa_bme) of the state the last step produced, before its balance."""
        out = (C.c_double * 2)()
        _chk(lib().gp_od_last_kappa(self._c, out), "gp_od_last_kappa")
        return out[0], out[1]

    def synchronize(self):
        _chk(lib().gp_synchronize(self._c), "gp_synchronize")

    def launch_counts(self):
        a, b = C.c_longlong(0), C.c_longlong(0)
        _chk(lib().gp_launch_counts(self._c, C.byref(a), C.byref(b)), "gp_launch_counts")
        return a.value, b.value

    def timing(self, on):
        _chk(lib().gp_timing_enable(self._c, 1 if on else 0), "gp_timing_enable")

    def timing_read(self):
        """{kernel name: (total ms, launches)} since timing was switched on."""
        m = 32
        n = C.c_int(0)
        names = (C.c_char_p * m)()
        ms = (C.c_double * m)()
        cnt = (C.c_longlong * m)()
        _chk(lib().gp_timing_read(self._c, m, C.byref(n), names, ms, cnt), "gp_timing_read")
        return {names[i].decode(): (ms[i], cnt[i]) for i in range(n.value)}
