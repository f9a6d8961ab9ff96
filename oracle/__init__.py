"""ctypes binding of liboracle.so — the CPU oracle.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package (see oracle/oracle.h).  It imports nothing from paper_1311_0861_b200.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

GAS, STARS = 1, 2
POISSON_NONE, POISSON_PERIODIC, POISSON_ISOLATED = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW = 0, 1
OK, ERR_ARG, ERR_ALLOC, ERR_STATE, ERR_UNSUPPORTED = 0, 1, 2, 5, 6
FIELDS = ["rho", "mx", "my", "mz", "E",
          "n", "nux", "nuy", "nuz", "Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz", "phi"]
OD_FIELDS = ["eps", "Pxx", "Pxy", "Pxz", "Pyy", "Pyz", "Pzz"]      # carried fields of the overdetermined system
FIELD_ID = {name: i for i, name in enumerate(FIELDS + OD_FIELDS)}
GAS_FIELDS = FIELDS[:5]
STAR_FIELDS = FIELDS[5:15]

_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int] * 3 + [C.c_double, C.c_int, C.c_int, C.c_double, C.c_double] + [C.c_int] * 3
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_threads.restype = C.c_int
        for name in ("orc_set_field", "orc_get_field", "orc_get_star_field"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int, _dp]
        for name in ("orc_eulerian", "orc_lagrangian", "orc_lagrangian_only", "orc_step"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_double]
        for name in ("orc_od_eulerian", "orc_od_lagrangian", "orc_od_lagrangian_only"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_double]
        L.orc_od_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.orc_od_enable.argtypes = [C.c_void_p]
        L.orc_od_balance.argtypes = [C.c_void_p]
        L.orc_kappa.argtypes = [C.c_void_p, _dp]
        L.orc_max_dt.argtypes = [C.c_void_p, C.c_double, _dp]
        L.orc_solve_poisson.argtypes = [C.c_void_p]
        L.orc_get_phi_padded.argtypes = [C.c_void_p, _dp]
        L.orc_gas_face.argtypes = [C.c_double] * 7 + [_dp, _dp]
        L.orc_gas_face.restype = None
        L.orc_bme_face.argtypes = [C.c_int, C.c_double, _dp, _dp, C.c_double, _dp, _dp, _dp, _dp]
        L.orc_bme_face.restype = None
        L.orc_fft1d.argtypes = [_dp, _dp, C.c_int, C.c_int]
        L.orc_poisson_direct.argtypes = [C.c_int] * 3 + [C.c_double, C.c_double, _dp] + [C.c_int] * 6 + [_dp]
        L.orc_kernel_self.restype = C.c_double
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"oracle: {what} failed with code {code}")
        self.code = code


def _chk(code, what):
    if code != OK:
        raise OracleError(code, what)


class Oracle:
    """One grid + state.  Arrays are numpy float64 of shape (nz, ny, nx) (x fastest)."""

    def __init__(self, nx, ny, nz, h, components=GAS, poisson=POISSON_NONE, G=1.0, gamma=5.0 / 3.0,
                 bc=(BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)):
        self.nx, self.ny, self.nz, self.h = nx, ny, nz, h
        self.components, self.poisson = components, poisson
        self.shape = (nz, ny, nx)
        self._c = lib().orc_create(nx, ny, nz, h, components, poisson, G, gamma, *bc)
        if not self._c:
            raise OracleError(ERR_ARG, "orc_create")

    def close(self):
        if self._c:
            lib().orc_destroy(self._c)
            self._c = None

    def __del__(self):
        self.close()

    def field_names(self):
        out = []
        if self.components & GAS:
            out += GAS_FIELDS
        if self.components & STARS:
            out += STAR_FIELDS
        return out

    def set(self, name, arr):
        a = np.ascontiguousarray(arr, dtype=np.float64)
        assert a.shape == self.shape, (a.shape, self.shape)
        _chk(lib().orc_set_field(self._c, FIELD_ID[name], _p(a)), f"set {name}")

    def set_state(self, state):
        for k, v in state.items():
            self.set(k, v)

    def get(self, name):
        out = np.empty(self.shape, dtype=np.float64)
        _chk(lib().orc_get_field(self._c, FIELD_ID[name], _p(out)), f"get {name}")
        return out

    def get_star(self, name):
        out = np.empty(self.shape, dtype=np.float64)
        _chk(lib().orc_get_star_field(self._c, FIELD_ID[name], _p(out)), f"get* {name}")
        return out

    def get_state(self):
        return {k: self.get(k) for k in self.field_names()}

    def phi_padded(self):
        out = np.empty((self.nz + 2, self.ny + 2, self.nx + 2), dtype=np.float64)
        _chk(lib().orc_get_phi_padded(self._c, _p(out)), "phi_padded")
        return out

    def eulerian(self, dt):
        _chk(lib().orc_eulerian(self._c, dt), "eulerian")

    def lagrangian(self, dt):
        _chk(lib().orc_lagrangian(self._c, dt), "lagrangian")

    def lagrangian_only(self, dt):
        _chk(lib().orc_lagrangian_only(self._c, dt), "lagrangian_only")

    def step(self, dt):
        _chk(lib().orc_step(self._c, dt), "step")

    def max_dt(self, cfl):
        dt = C.c_double(0.0)
        _chk(lib().orc_max_dt(self._c, cfl, C.byref(dt)), "max_dt")
        return dt.value

    def solve_poisson(self):
        _chk(lib().orc_solve_poisson(self._c), "solve_poisson")

    # ---- overdetermined system (PAPER.md:41 4th equation, 65, 194-202) ----
    def od_enable(self):
        _chk(lib().orc_od_enable(self._c), "od_enable")

    def od_field_names(self):
        return (["eps"] if self.components & GAS else []) + (OD_FIELDS[1:] if self.components & STARS else [])

    def od_eulerian(self, dt):
        _chk(lib().orc_od_eulerian(self._c, dt), "od_eulerian")

    def od_lagrangian_only(self, dt):
        _chk(lib().orc_od_lagrangian_only(self._c, dt), "od_lagrangian_only")

    def od_step(self, dt, balance=True):
        _chk(lib().orc_od_step(self._c, dt, 1 if balance else 0), "od_step")

    def od_balance(self):
        _chk(lib().orc_od_balance(self._c), "od_balance")

    def kappa(self):
        out = np.zeros(2)
        _chk(lib().orc_kappa(self._c, _p(out)), "kappa")
        return float(out[0]), float(out[1])


def gas_face(gamma, rhoL, vL, pL, rhoR, vR, pR):
    V, P = C.c_double(), C.c_double()
    lib().orc_gas_face(gamma, rhoL, vL, pL, rhoR, vR, pR, C.byref(V), C.byref(P))
    return V.value, P.value


def bme_face(d, nL, uL, PiL, nR, uR, PiR):
    uL, PiL, uR, PiR = (np.ascontiguousarray(x, dtype=np.float64) for x in (uL, PiL, uR, PiR))
    us, Pid = np.empty(3), np.empty(3)
    lib().orc_bme_face(d, nL, _p(uL), _p(PiL), nR, _p(uR), _p(PiR), _p(us), _p(Pid))
    return us, Pid


def fft1d(x, sign=-1):
    x = np.asarray(x, dtype=np.complex128)
    re, im = np.ascontiguousarray(x.real), np.ascontiguousarray(x.imag)
    _chk(lib().orc_fft1d(_p(re), _p(im), len(re), sign), "fft1d")
    return re + 1j * im


def poisson_direct(dens, h, G=1.0, lo=None, hi=None):
    """Direct summation of the isolated potential over the index box [lo, hi) (z, y, x order)."""
    dens = np.ascontiguousarray(dens, dtype=np.float64)
    nz, ny, nx = dens.shape
    lo = lo or (0, 0, 0)
    hi = hi or (nz, ny, nx)
    out = np.empty((hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]))
    _chk(lib().orc_poisson_direct(nx, ny, nz, h, G, _p(dens), lo[2], hi[2], lo[1], hi[1], lo[0], hi[0], _p(out)),
         "poisson_direct")
    return out


def kernel_self():
    return lib().orc_kernel_self()


def set_threads(n):
    lib().orc_set_threads(int(n))


def get_threads():
    return lib().orc_get_threads()
