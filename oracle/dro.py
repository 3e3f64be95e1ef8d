"""ctypes binding of the CPU oracle (oracle/dro.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It shares nothing with the CUDA path.
Argument marshalling only; all arithmetic is in dro.cpp (which cites the paper).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dro.cpp")
_LIB = os.path.join(_HERE, "libdro.so")

OK, ERR_ARG, ERR_WORKSPACE, ERR_CUDA, ERR_DIVERGED, ERR_STATE, MAXITER = range(7)
CFL, ST_FACTOR, NCHECK, GAVG, VOID_REL, BC_MODE = range(6)
FORM = 8
STAG_TOL = 10
STOP_NONE, STOP_RESIDUAL, STOP_STAGNATION, STOP_MAXITER = range(4)
FIELDS = ("vx", "vy", "vz", "sxx", "syy", "szz", "tyz", "txz", "txy")


def build(force: bool = False) -> str:
    """Compile oracle/dro.cpp -> oracle/libdro.so with g++ (plain -O2, OpenMP on the outer z loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++17", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.dro_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, dp, dp, C.POINTER(C.c_void_p)]
        L.dro_set_param.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.dro_solve.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int]
        L.dro_step.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int]
        L.dro_iterate.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int]
        L.dro_effective_C.argtypes = [C.c_void_p, dp]
        L.dro_avg_stress.argtypes = [C.c_void_p, dp]
        L.dro_offdiag_direct.argtypes = [C.c_void_p, dp]
        L.dro_info.argtypes = [C.c_void_p, C.POINTER(C.c_int), dp, dp]
        L.dro_field_size.argtypes = [C.c_void_p, C.c_int]
        L.dro_field_size.restype = C.c_size_t
        L.dro_get_field.argtypes = [C.c_void_p, C.c_int, dp, C.c_size_t]
        L.dro_last_error.argtypes = [C.c_void_p]
        L.dro_last_error.restype = C.c_char_p
        L.dro_stop_reason.argtypes = [C.c_void_p]
        L.dro_raw_size.argtypes = [C.c_void_p, C.c_int]
        L.dro_raw_size.restype = C.c_size_t
        L.dro_get_raw.argtypes = [C.c_void_p, C.c_int, dp, C.c_size_t]
        L.dro_set_raw.argtypes = [C.c_void_p, C.c_int, dp, C.c_size_t]
        L.dro_destroy.argtypes = [C.c_void_p]
        L.dro_destroy.restype = None
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class OracleError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("dro status %d: %s" % (status, msg))
        self.status = status


class Oracle:
    """K, G: numpy arrays of shape (nz, ny, nx) (x fastest in memory), fp64."""

    def __init__(self, K, G, h=1.0, **params):
        K = np.ascontiguousarray(K, dtype=np.float64)
        G = np.ascontiguousarray(G, dtype=np.float64)
        assert K.ndim == 3 and K.shape == G.shape
        self.nz, self.ny, self.nx = K.shape
        self._h = C.c_void_p()
        st = lib().dro_create(self.nx, self.ny, self.nz, float(h), _dp(K), _dp(G), C.byref(self._h))
        if st != OK:
            raise OracleError(st, "dro_create rejected its arguments")
        for k, v in params.items():
            self.set_param(k, v)

    def _check(self, st, soft=(OK,)):
        if st not in soft:
            raise OracleError(st, lib().dro_last_error(self._h).decode())
        return st

    def set_param(self, name, value):
        ids = dict(cfl=CFL, st_factor=ST_FACTOR, ncheck=NCHECK, gavg=GAVG, void_rel=VOID_REL, bc_mode=BC_MODE, form=FORM, stag_tol=STAG_TOL)
        self._check(lib().dro_set_param(self._h, ids[name], float(value)))

    def solve(self, lc, eps0=1e-4, tol=1e-8, maxiter=100000):
        return self._check(lib().dro_solve(self._h, lc, eps0, tol, maxiter), soft=(OK, MAXITER))

    def step(self, lc, eps0, niter):
        return self._check(lib().dro_step(self._h, lc, eps0, niter))

    def iterate(self, lc, eps0, niter):
        return self._check(lib().dro_iterate(self._h, lc, eps0, niter))

    def effective_C(self):
        out = np.zeros(36)
        self._check(lib().dro_effective_C(self._h, _dp(out)))
        return out.reshape(6, 6)

    def avg_stress(self):
        out = np.zeros(6)
        self._check(lib().dro_avg_stress(self._h, _dp(out)))
        return out

    def offdiag_direct(self):
        """(C12, C13, C23) by Eq. 27-29 from the triaxial test (load case 6) and C11, C22, C33 of load cases 0-2"""
        out = np.zeros(3)
        self._check(lib().dro_offdiag_direct(self._h, _dp(out)))
        return out

    def info(self):
        it = C.c_int()
        r = C.c_double()
        ms = C.c_double()
        lib().dro_info(self._h, C.byref(it), C.byref(r), C.byref(ms))
        return it.value, r.value, ms.value

    def stop_reason(self):
        return lib().dro_stop_reason(self._h)

    def field_shape(self, f):
        nx, ny, nz = self.nx, self.ny, self.nz
        return {0: (nz, ny, nx + 1), 1: (nz, ny + 1, nx), 2: (nz + 1, ny, nx),
                3: (nz, ny, nx), 4: (nz, ny, nx), 5: (nz, ny, nx),
                6: (nz + 1, ny + 1, nx), 7: (nz + 1, ny, nx + 1), 8: (nz, ny + 1, nx + 1)}[f]

    def get_field(self, f):
        if isinstance(f, str):
            f = FIELDS.index(f)
        out = np.empty(self.field_shape(f))
        self._check(lib().dro_get_field(self._h, f, _dp(out), out.size))
        return out

    RAW = ("vx", "vy", "vz", "p", "txx", "tyy", "tzz", "tyz", "txz", "txy")

    def raw_shape(self, name):
        return self.field_shape({"vx": 0, "vy": 1, "vz": 2, "p": 3, "txx": 3, "tyy": 3, "tzz": 3, "tyz": 6, "txz": 7, "txy": 8}[name])

    def get_raw(self, name):
        """the oracle's own state array (p and tau_aa separately, Eq. 10), for the z-slab halo test"""
        out = np.empty(self.raw_shape(name))
        self._check(lib().dro_get_raw(self._h, self.RAW.index(name), _dp(out), out.size))
        return out

    def set_raw(self, name, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == self.raw_shape(name)
        self._check(lib().dro_set_raw(self._h, self.RAW.index(name), _dp(a), a.size))

    def solve_all(self, eps0=1e-4, tol=1e-8, maxiter=100000):
        """six load cases -> (C[6,6], [(status, iters, residual)]*6)"""
        log = []
        for lc in range(6):
            st = self.solve(lc, eps0, tol, maxiter)
            it, r, _ = self.info()
            log.append((st, it, r))
        return self.effective_C(), log

    def close(self):
        if self._h:
            lib().dro_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
