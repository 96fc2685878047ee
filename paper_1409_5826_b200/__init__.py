"""paper_1409_5826_b200 -- thin Python binding of the C ABI in include/kinnet.h.

Argument marshalling only: every step of the hot path (rates, fluxes, F+/F-
sums, asymptotic/Euler update, dt control) runs in the sm_100a kernels of
csrc/kinnet.cu.  PyTorch supplies device memory and streams.  There is no CPU
fallback: if libkinnet.so is missing or cannot be loaded, importing the binding
raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkinnet.so")

NET_OK, NET_EINVAL, NET_ENOMEM, NET_ECUDA = 0, -1, -2, -3
NET_STATUS_MAX_STEPS, NET_STATUS_NONFINITE = 1, 2
NET_STATIC_MAX_ZONES = 65536  # largest batch of net_integrate_static (include/kinnet.h)

EXPORTS = (
    "net_default_params", "net_create", "net_create_host", "net_destroy", "net_integrate",
    "net_integrate_fixed", "net_integrate_host", "net_integrate_host_async", "net_wait", "net_reserve",
    "net_set_binding_energy", "net_integrate_energy", "net_rates", "net_rhs", "net_schedule_info",
    "net_schedule_table", "net_last_error", "net_integrate_static", "net_launch_stats",
)


class net_params_t(C.Structure):
    _fields_ = [
        ("kappa", C.c_double), ("eps_y", C.c_double), ("y_floor", C.c_double),
        ("growth", C.c_double), ("max_steps", C.c_longlong), ("precision", C.c_int),
        ("kernel", C.c_int), ("host_chunk", C.c_int), ("method", C.c_int),
    ]


class net_schedule_info_t(C.Structure):
    _fields_ = [(k, C.c_int) for k in (
        "n_species", "n_reactions", "threads", "flux_slots", "slots_2body", "slots_3body",
        "n_entries", "n_big_species", "n_entries_big", "small_max", "readback_max", "smem_bytes",
        "zones_per_sm", "kernel", "pull_ok", "pull_hubs", "pull_slots", "pull_slots2",
        "pull_agg_max", "pull_wavefronts", "pull_wavefronts_ideal", "pull_threads", "pull_nslots",
        "pull_stair")]


class KinnetError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"kinnet error {code}: {msg}")
        self.code = code


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python paper_1409_5826_b200/build.py` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
    create_args = [C.POINTER(vp), C.c_int, ip, C.c_int, ip, ip, ip, ip, dp, C.POINTER(net_params_t)]
    lib.net_default_params.argtypes = [C.POINTER(net_params_t)]
    lib.net_create.argtypes = create_args
    lib.net_create_host.argtypes = create_args
    lib.net_destroy.argtypes = [vp]
    lib.net_destroy.restype = None
    lib.net_integrate.argtypes = [vp, C.c_int, vp, vp, vp, C.c_double, vp, vp, vp, vp]
    lib.net_integrate_static.argtypes = [vp, C.c_int, vp, vp, vp, C.c_double, vp, vp, vp, vp]
    lib.net_set_binding_energy.argtypes = [vp, dp]
    lib.net_integrate_energy.argtypes = [vp, C.c_int, vp, vp, vp, C.c_double, vp, vp, vp, vp, vp]
    lib.net_integrate_fixed.argtypes = [vp, C.c_int, vp, vp, vp, C.c_double, C.c_longlong, vp]
    lib.net_integrate_host.argtypes = [vp, C.c_int, vp, vp, vp, C.c_double, vp, vp, vp]
    lib.net_integrate_host_async.argtypes = [vp, C.c_int, vp, vp, vp, C.c_double, vp, vp, vp]
    lib.net_wait.argtypes = [vp]
    lib.net_reserve.argtypes = [vp, C.c_int]
    lib.net_launch_stats.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), ip]
    lib.net_rates.argtypes = [vp, C.c_int, vp, vp, vp, vp]
    lib.net_rhs.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp]
    lib.net_schedule_info.argtypes = [vp, C.POINTER(net_schedule_info_t)]
    lib.net_schedule_table.argtypes = [vp, C.c_char_p, ip, C.c_int]
    lib.net_last_error.restype = C.c_char_p
    return lib


lib = _load()


def net_last_error() -> str:
    return lib.net_last_error().decode()


def _check(rc: int) -> int:
    if rc < 0:
        raise KinnetError(rc, net_last_error())
    return rc


@dataclass
class NetParams:
    kappa: float = 1.0
    eps_y: float = 0.05
    y_floor: float = 1e-10
    growth: float = 2.0
    max_steps: int = 10_000_000
    precision: int = 64
    kernel: int = 0  # 0 = automatic, 1 = generic kernel only, 2 = one-species pull kernel
    host_chunk: int = 0  # staged host path: zones per chunk; < 0 = never zero-copy
    method: int = 0  # 0 = asymptotic (the paper's method), 1 = QSS variant

    def to_c(self) -> net_params_t:
        return net_params_t(self.kappa, self.eps_y, self.y_floor, self.growth, self.max_steps,
                            self.precision, self.kernel, self.host_chunk, self.method)


def net_default_params() -> NetParams:
    p = net_params_t()
    _check(lib.net_default_params(C.byref(p)))
    return NetParams(p.kappa, p.eps_y, p.y_floor, p.growth, p.max_steps, p.precision, p.kernel, p.host_chunk, p.method)


def _ptr(t):
    """Device (torch tensor) or host (numpy array) address, None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch

        stream = torch.cuda.current_stream()
    return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))


class Net:
    """Owner of one net_t.  ``net`` needs A, n_react, react, n_prod, prod, coef."""

    def __init__(self, net, params: NetParams | None = None, host_only: bool = False):
        self.params = params or NetParams()
        self.N = int(len(net.A))
        self.M = int(len(net.n_react))
        A = np.ascontiguousarray(net.A, np.int32)
        nr = np.ascontiguousarray(net.n_react, np.int32)
        re = np.ascontiguousarray(net.react, np.int32).reshape(-1)
        npd = np.ascontiguousarray(net.n_prod, np.int32)
        pr = np.ascontiguousarray(net.prod, np.int32).reshape(-1)
        co = np.ascontiguousarray(net.coef, np.float64).reshape(-1)
        ip, dp = C.POINTER(C.c_int), C.POINTER(C.c_double)
        h = C.c_void_p()
        cp = self.params.to_c()
        fn = lib.net_create_host if host_only else lib.net_create
        _check(fn(C.byref(h), self.N, A.ctypes.data_as(ip), self.M, nr.ctypes.data_as(ip),
                  re.ctypes.data_as(ip), npd.ctypes.data_as(ip), pr.ctypes.data_as(ip),
                  co.ctypes.data_as(dp), C.byref(cp)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None) and lib is not None:
            lib.net_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    @property
    def handle(self):
        return self._h

    def schedule_info(self) -> dict:
        info = net_schedule_info_t()
        _check(lib.net_schedule_info(self._h, C.byref(info)))
        return {k: getattr(info, k) for k, _ in info._fields_}

    def schedule_table(self, name: str) -> np.ndarray:
        n = _check(lib.net_schedule_table(self._h, name.encode(), None, 0))
        out = np.zeros(max(n, 1), np.int32)
        _check(lib.net_schedule_table(self._h, name.encode(), out.ctypes.data_as(C.POINTER(C.c_int)), n))
        return out[:n]

    # ---- the calls of include/kinnet.h, same names, same argument order ----
    def net_integrate(self, zones, T9, rho, Y, t_hydro, dt=None, n_steps=None, status=None,
                      stream=None):
        _check(lib.net_integrate(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y), float(t_hydro),
                                 _ptr(dt), _ptr(n_steps), _ptr(status), _stream(stream)))

    def net_integrate_static(self, zones, T9, rho, Y, t_hydro, dt=None, n_steps=None, status=None,
                             stream=None):
        """net_integrate without any device allocation behind it, for callers that may not
        allocate while they run (their own pool owns the GPU's memory, or they sit in a region
        where cudaMalloc is illegal): the launch-order scratch is a fixed 264 KB array in the
        library.  At most NET_STATIC_MAX_ZONES zones per call; one call at a time per device
        (calls that overlap on the GPU race on the array); make the first call on a device
        before any stream capture.  Same arguments and bit-identical results (include/kinnet.h)."""
        _check(lib.net_integrate_static(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y),
                                        float(t_hydro), _ptr(dt), _ptr(n_steps), _ptr(status),
                                        _stream(stream)))

    def net_set_binding_energy(self, B):
        B = np.ascontiguousarray(B, np.float64)
        assert B.shape == (self.N,)
        _check(lib.net_set_binding_energy(self._h, B.ctypes.data_as(C.POINTER(C.c_double))))

    def net_integrate_energy(self, zones, T9, rho, Y, t_hydro, dt=None, n_steps=None, status=None,
                             energy=None, stream=None):
        _check(lib.net_integrate_energy(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y),
                                        float(t_hydro), _ptr(dt), _ptr(n_steps), _ptr(status),
                                        _ptr(energy), _stream(stream)))

    def net_integrate_fixed(self, zones, T9, rho, Y, dt_fixed, n_steps, stream=None):
        _check(lib.net_integrate_fixed(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y),
                                       float(dt_fixed), int(n_steps), _stream(stream)))

    def net_integrate_host(self, zones, T9, rho, Y, t_hydro, dt=None, n_steps=None, status=None):
        _check(lib.net_integrate_host(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y),
                                      float(t_hydro), _ptr(dt), _ptr(n_steps), _ptr(status)))

    def net_integrate_host_async(self, zones, T9, rho, Y, t_hydro, dt=None, n_steps=None, status=None):
        _check(lib.net_integrate_host_async(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y),
                                            float(t_hydro), _ptr(dt), _ptr(n_steps), _ptr(status)))

    def net_wait(self):
        _check(lib.net_wait(self._h))

    def net_reserve(self, max_zones):
        _check(lib.net_reserve(self._h, int(max_zones)))

    def net_launch_stats(self) -> dict:
        a, b, c = C.c_longlong(), C.c_longlong(), C.c_int()
        _check(lib.net_launch_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return {"sorted_calls": a.value, "unsorted_calls": b.value, "lanes_pinned": c.value}

    def net_rates(self, zones, T9, rho, R, stream=None):
        _check(lib.net_rates(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(R), _stream(stream)))

    def net_rhs(self, zones, T9, rho, Y, Fplus, Fminus, stream=None):
        _check(lib.net_rhs(self._h, int(zones), _ptr(T9), _ptr(rho), _ptr(Y), _ptr(Fplus),
                           _ptr(Fminus), _stream(stream)))
