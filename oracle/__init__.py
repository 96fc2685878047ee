"""ctypes face of the CPU oracle (oracle/asym_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  Nothing under
paper_1409_5826_b200/ imports this, and this imports nothing from there.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from .build import build

_I = C.POINTER(C.c_int)
_D = C.POINTER(C.c_double)
_L = C.POINTER(C.c_longlong)


class _Params(C.Structure):
    _fields_ = [
        ("kappa", C.c_double),
        ("eps_y", C.c_double),
        ("y_floor", C.c_double),
        ("growth", C.c_double),
        ("max_steps", C.c_longlong),
        ("method", C.c_int),
    ]


@dataclass
class OracleParams:
    kappa: float = 1.0
    eps_y: float = 0.05
    y_floor: float = 1e-10
    growth: float = 2.0
    max_steps: int = 10_000_000
    method: int = 0  # 0 = asymptotic (the paper's method), 1 = QSS variant


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.oracle_create.restype = C.c_void_p
        lib.oracle_create.argtypes = [C.c_int, _I, C.c_int, _I, _I, _I, _I, _D, C.POINTER(_Params)]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_num_edges.argtypes = [C.c_void_p]
        lib.oracle_rates.argtypes = [C.c_void_p, C.c_double, C.c_double, _D]
        lib.oracle_rates_ld.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        lib.oracle_rhs.argtypes = [C.c_void_p, _D, _D, _D, _D, _D]
        lib.oracle_integrate.argtypes = [
            C.c_void_p, C.c_int, _D, _D, C.c_void_p, C.c_double, _D, _L, _I, _L, C.c_int, C.c_int,
        ]
        lib.oracle_integrate_fixed.argtypes = [
            C.c_void_p, C.c_int, _D, _D, C.c_void_p, C.c_double, C.c_longlong, _L, C.c_int, C.c_int,
        ]
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def _ip(a):
    return a.ctypes.data_as(_I)


def _dp(a):
    return a.ctypes.data_as(_D)


class Oracle:
    """One network compiled for the oracle (O1).  ``net`` needs the attributes
    A, n_react, react, n_prod, prod, coef (see gen.Network)."""

    def __init__(self, net, params: OracleParams | None = None):
        lib = _load()
        self.N = int(len(net.A))
        self.M = int(len(net.n_react))
        self._keep = [
            np.ascontiguousarray(net.A, np.int32),
            np.ascontiguousarray(net.n_react, np.int32),
            np.ascontiguousarray(net.react, np.int32).reshape(-1),
            np.ascontiguousarray(net.n_prod, np.int32),
            np.ascontiguousarray(net.prod, np.int32).reshape(-1),
            np.ascontiguousarray(net.coef, np.float64).reshape(-1),
        ]
        p = params or OracleParams()
        cp = _Params(p.kappa, p.eps_y, p.y_floor, p.growth, p.max_steps, p.method)
        A, nr, re, npd, pr, co = self._keep
        self._h = lib.oracle_create(self.N, _ip(A), self.M, _ip(nr), _ip(re), _ip(npd), _ip(pr),
                                    _dp(co), C.byref(cp))
        if not self._h:
            raise ValueError("oracle_create rejected the tables")
        self.A = A.astype(np.float64)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.oracle_destroy(self._h)
            self._h = None

    @property
    def n_edges(self) -> int:
        return int(_lib.oracle_num_edges(self._h))

    def rates(self, T9: float, rho: float) -> np.ndarray:
        R = np.empty(self.M, np.float64)
        _lib.oracle_rates(self._h, float(T9), float(rho), _dp(R))
        return R

    def rates_ld(self, T9: float, rho: float) -> np.ndarray:
        """O2 as the long-double arbiter evaluates it (np.longdouble, x87 extended)."""
        assert np.dtype(np.longdouble).itemsize == C.sizeof(C.c_longdouble)
        R = np.empty(self.M, np.longdouble)
        _lib.oracle_rates_ld(self._h, float(T9), float(rho), R.ctypes.data_as(C.c_void_p))
        return R

    def rhs(self, R, Y):
        """(f, F+, F-) for one state (double)."""
        R = np.ascontiguousarray(R, np.float64)
        Y = np.ascontiguousarray(Y, np.float64)
        f = np.empty(self.M)
        Fp = np.empty(self.N)
        Fm = np.empty(self.N)
        _lib.oracle_rhs(self._h, _dp(R), _dp(Y), _dp(f), _dp(Fp), _dp(Fm))
        return f, Fp, Fm

    def _state(self, Y, precision):
        dt = np.float32 if precision == 32 else np.float64  # 64, and 80 (the long-double arbiter)
        Y = np.array(Y, dtype=dt, order="C", copy=True)
        if Y.ndim == 1:
            Y = Y[None, :]
        assert Y.shape[1] == self.N
        return Y

    def integrate(self, T9, rho, Y, t_hydro, dt=None, precision=64, n_threads=1):
        """One hydro step, adaptive dt.  Returns dict(Y, dt, n_steps, status, n_asym)."""
        Y = self._state(Y, precision)
        z = Y.shape[0]
        T9 = np.ascontiguousarray(np.broadcast_to(np.asarray(T9, np.float64), (z,)))
        rho = np.ascontiguousarray(np.broadcast_to(np.asarray(rho, np.float64), (z,)))
        dt_io = np.zeros(z) if dt is None else np.array(dt, np.float64, copy=True).reshape(z)
        n_steps = np.zeros(z, np.int64)
        status = np.zeros(z, np.int32)
        n_asym = np.zeros(z, np.int64)
        rc = _lib.oracle_integrate(
            self._h, z, _dp(T9), _dp(rho), Y.ctypes.data_as(C.c_void_p), float(t_hydro),
            _dp(dt_io), n_steps.ctypes.data_as(_L), _ip(status), n_asym.ctypes.data_as(_L),
            int(precision), int(n_threads),
        )
        assert rc == 0
        return dict(Y=Y, dt=dt_io, n_steps=n_steps, status=status, n_asym=n_asym)

    @staticmethod
    def energy(B, Y0, Y):
        """Integrated energy release per zone (reading Q19), the
        definition written out in fp64: E_z = sum_i B_i * (Y_i(t_hydro) - Y_i(0))."""
        B = np.asarray(B, np.float64)
        Y0 = np.atleast_2d(np.asarray(Y0, np.float64))
        Y = np.atleast_2d(np.asarray(Y, np.float64))
        E = np.zeros(Y.shape[0])
        for z in range(Y.shape[0]):
            for i in range(Y.shape[1]):  # species order
                E[z] += B[i] * (Y[z, i] - Y0[z, i])
        return E

    def integrate_fixed(self, T9, rho, Y, dt_fixed, n_steps, precision=64, n_threads=1):
        """Exactly n_steps sub-steps of dt_fixed.  Returns dict(Y, n_asym)."""
        Y = self._state(Y, precision)
        z = Y.shape[0]
        T9 = np.ascontiguousarray(np.broadcast_to(np.asarray(T9, np.float64), (z,)))
        rho = np.ascontiguousarray(np.broadcast_to(np.asarray(rho, np.float64), (z,)))
        n_asym = np.zeros(z, np.int64)
        rc = _lib.oracle_integrate_fixed(
            self._h, z, _dp(T9), _dp(rho), Y.ctypes.data_as(C.c_void_p), float(dt_fixed),
            int(n_steps), n_asym.ctypes.data_as(_L), int(precision), int(n_threads),
        )
        assert rc == 0
        return dict(Y=Y, n_asym=n_asym)
