"""ctypes driver for ``hydro_oracle.c`` (argument marshalling only; no arithmetic here).

Test infrastructure: see the header of ``hydro_oracle.c``.  ``build()`` compiles the C file
with ``-O2 -ffp-contract=off`` (oracle/Makefile) the first time it is needed.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_hydro.so")
_SRC = os.path.join(_HERE, "hydro_oracle.c")

BC_OUTFLOW, BC_REFLECT, BC_PERIODIC = 0, 1, 2
_ERR = {1: "ERR_ARG", 2: "ERR_ALLOC", 4: "ERR_UNPHYSICAL", 5: "ERR_NOSTATE"}


class OracleError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"oracle {where}: {_ERR.get(code, code)}")
        self.code = code


def build(force=False):
    """Compile liboracle_hydro.so next to its source if missing or stale."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
        return _SO
    subprocess.run(["make", "-C", _HERE, "-B", "liboracle_hydro.so"], check=True,
                   stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
    return _SO


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp = C.c_void_p
        L.oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                    C.POINTER(C.c_int), C.POINTER(vp)]
        L.oracle_create_nd.argtypes = [C.c_int, C.POINTER(C.c_int), _dp, C.c_double,
                                       C.POINTER(C.c_int), C.POINTER(vp)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_set_state.argtypes = [vp, _dp]
        L.oracle_get_state.argtypes = [vp, _dp]
        L.oracle_get_padded.argtypes = [vp, _dp]
        L.oracle_ghost_fill.argtypes = [vp]
        L.oracle_cfl_dt.argtypes = [vp, _dp]
        L.oracle_max_signal_speed.argtypes = [vp, _dp]
        L.oracle_step.argtypes = [vp, C.c_double]
        L.oracle_evolve.argtypes = [vp, C.c_double, C.POINTER(C.c_longlong)]
        L.oracle_set_cfl.argtypes = [vp, C.c_double]
        L.oracle_set_limiter_theta.argtypes = [vp, C.c_double]
        L.oracle_get_time.argtypes = [vp, _dp, C.POINTER(C.c_longlong)]
        L.oracle_set_threads.argtypes = [C.c_int]
        L.oracle_get_threads.restype = C.c_int
        L.oracle_sum3.argtypes = [C.c_double] * 3
        L.oracle_sum3.restype = C.c_double
        L.oracle_minmod.argtypes = [C.c_double] * 3
        L.oracle_minmod.restype = C.c_double
        L.oracle_primitive.argtypes = [C.c_double, _dp, _dp]
        L.oracle_primitive.restype = None
        L.oracle_hll_flux.argtypes = [C.c_double, C.c_int, _dp, _dp, _dp]
        L.oracle_hll_flux.restype = None
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(_dp)


def sum3(a, b, c):
    return lib().oracle_sum3(a, b, c)


def minmod(theta, a, b):
    return lib().oracle_minmod(theta, a, b)


def primitive(gamma, U):
    U = np.ascontiguousarray(U, dtype=np.float64)
    W = np.empty(5)
    lib().oracle_primitive(gamma, _ptr(U), _ptr(W))
    return W


def hll_flux(gamma, d, WL, WR):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.empty(5)
    lib().oracle_hll_flux(gamma, d, _ptr(WL), _ptr(WR), _ptr(F))
    return F


def set_threads(n):
    rc = lib().oracle_set_threads(int(n))
    if rc:
        raise OracleError(rc, "set_threads")


def get_threads():
    return lib().oracle_get_threads()


class OracleHydro:
    """Same call names as the C-ABI of the product (``include/hydro.h``), oracle side."""

    def __init__(self, nx, ny, nz, gamma, dx, bc, ndim=None, dxyz=None):
        """3D run with cubic cells (oracle_create) or, with `ndim` given, a run of dimension ndim
        with cell edges `dxyz` (oracle_create_nd; extents of inactive axes must be 1)."""
        self.shape = (5, nz, ny, nx)
        self._h = C.c_void_p()
        arr = (C.c_int * 6)(*[int(b) for b in bc])
        if ndim is None:
            self.padded_shape = (5, nz + 4, ny + 4, nx + 4)
            self._chk(lib().oracle_create(nx, ny, nz, gamma, dx, arr, C.byref(self._h)), "create")
        else:
            g = [4 if a < ndim else 0 for a in range(3)]
            self.padded_shape = (5, nz + g[2], ny + g[1], nx + g[0])
            n = (C.c_int * 3)(nx, ny, nz)
            d = (C.c_double * 3)(*(dxyz if dxyz is not None else (dx, dx, dx)))
            self._chk(lib().oracle_create_nd(ndim, n, d, gamma, arr, C.byref(self._h)), "create_nd")

    @staticmethod
    def _chk(rc, where):
        if rc:
            raise OracleError(rc, where)

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_cfl(self, cfl):
        self._chk(lib().oracle_set_cfl(self._h, cfl), "set_cfl")

    def set_limiter_theta(self, theta):
        self._chk(lib().oracle_set_limiter_theta(self._h, theta), "set_limiter_theta")

    def set_state(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == self.shape, (U.shape, self.shape)
        self._chk(lib().oracle_set_state(self._h, _ptr(U)), "set_state")

    def get_state(self):
        U = np.empty(self.shape)
        self._chk(lib().oracle_get_state(self._h, _ptr(U)), "get_state")
        return U

    def get_padded(self):
        U = np.empty(self.padded_shape)
        self._chk(lib().oracle_get_padded(self._h, _ptr(U)), "get_padded")
        return U

    def ghost_fill(self):
        self._chk(lib().oracle_ghost_fill(self._h), "ghost_fill")

    def cfl_dt(self):
        dt = C.c_double()
        self._chk(lib().oracle_cfl_dt(self._h, C.byref(dt)), "cfl_dt")
        return dt.value

    def max_signal_speed(self):
        s = C.c_double()
        self._chk(lib().oracle_max_signal_speed(self._h, C.byref(s)), "max_signal_speed")
        return s.value

    def step(self, dt):
        self._chk(lib().oracle_step(self._h, dt), "step")

    def evolve(self, t_final):
        n = C.c_longlong()
        self._chk(lib().oracle_evolve(self._h, t_final, C.byref(n)), "evolve")
        return n.value

    def get_time(self):
        t, n = C.c_double(), C.c_longlong()
        self._chk(lib().oracle_get_time(self._h, C.byref(t), C.byref(n)), "get_time")
        return t.value, n.value
