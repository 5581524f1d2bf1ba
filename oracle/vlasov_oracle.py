"""ctypes front end of ``vlasov_oracle.c`` (TEST INFRASTRUCTURE, see __init__).

No arithmetic of the method happens here: arrays are passed to the C oracle
and results are returned as numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vlasov_oracle.c")
_LIB = os.path.join(_HERE, "libvlasov_oracle.so")

MODEL_FREE, MODEL_HMF, MODEL_RING, MODEL_SHEET = 0, 1, 2, 3
BC_PERIODIC, BC_ZERO = 0, 1
KEY_EPS, KEY_PRECISION, KEY_BC_X, KEY_BC_P, KEY_HISTORY, KEY_SPLINE, KEY_ORDER = 1, 2, 3, 4, 5, 6, 7
SPLINE_FD, SPLINE_GS = 0, 1
GS_EXT = 64

_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, OpenMP) if missing or stale."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_dp = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            lib.oracle_init.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_int), _dp, ctypes.c_double]
            lib.oracle_set_param.argtypes = [ctypes.c_int, ctypes.c_double]
            lib.oracle_upload.argtypes = [_dp]
            lib.oracle_download.argtypes = [_dp]
            lib.oracle_step.argtypes = [ctypes.c_int]
            lib.oracle_moments.argtypes = [_dp]
            lib.oracle_casimirs.argtypes = [_dp]
            lib.oracle_density.argtypes = [_dp]
            lib.oracle_force.argtypes = [_dp]
            lib.oracle_theta_sweep.argtypes = [ctypes.c_double]
            lib.oracle_p_sweep.argtypes = [ctypes.c_double]
            lib.oracle_p_sweep_with_force.argtypes = [_dp, ctypes.c_double]
            lib.oracle_free.restype = None
            lib.oracle_set_threads.argtypes = [ctypes.c_int]
            lib.oracle_set_threads.restype = None
            lib.oracle_get_threads.restype = ctypes.c_int
            lib.oracle_fd8_second_derivative.argtypes = [_dp, ctypes.c_long, ctypes.c_double, ctypes.c_int, _dp]
            lib.oracle_fd8_second_derivative.restype = None
            lib.oracle_shift_line_alloc.argtypes = [_dp, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_int, _dp]
            lib.oracle_gs_second_derivative.argtypes = [_dp, ctypes.c_long, ctypes.c_double, ctypes.c_int, _dp]
            lib.oracle_shift_line_kind_alloc.argtypes = [_dp, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int, _dp]
            lib.oracle_force_from_rho.argtypes = [ctypes.c_int, _dp, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double, _dp]
            lib.oracle_force_from_rho.restype = None
            _lib = lib
    return _lib


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError("oracle %s failed with code %d" % (what, rc))


# ---- stateless line-level entry points (used by the pins) -------------------

def fd8_second_derivative(u, h: float, bc: int = BC_PERIODIC) -> np.ndarray:
    """eq (16).  Periodic: n values.  Zero extension: n+10 values for k=-5..n+4."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    n = u.shape[0]
    out = np.empty(n if bc == BC_PERIODIC else n + 10, dtype=np.float64)
    _load().oracle_fd8_second_derivative(_ptr(u), n, float(h), int(bc), _ptr(out))
    return out


def gs_second_derivative(u, h: float, bc: int = BC_PERIODIC) -> np.ndarray:
    """System (15).  Periodic: n values.  Zero extension: n+128 values for k=-64..n+63."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    n = u.shape[0]
    out = np.empty(n if bc == BC_PERIODIC else n + 2 * GS_EXT, dtype=np.float64)
    _check(_load().oracle_gs_second_derivative(_ptr(u), n, float(h), int(bc), _ptr(out)), "gs_second_derivative")
    return out


def shift_line(u, h: float, disp: float, bc: int = BC_PERIODIC, spline: int = SPLINE_FD) -> np.ndarray:
    """out_i = f(x_i - disp) by eqs (13)-(14) with f'' from eq (16) (or system (15) for SPLINE_GS)."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.empty_like(u)
    _check(_load().oracle_shift_line_kind_alloc(_ptr(u), u.shape[0], float(h), float(disp), int(bc), int(spline),
                                                _ptr(out)), "shift_line")
    return out


def force_from_rho(model: int, rho, xmin: float, xmax: float, eps: float = 0.01) -> np.ndarray:
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    out = np.empty_like(rho)
    _load().oracle_force_from_rho(int(model), _ptr(rho), rho.shape[0], float(xmin), float(xmax), float(eps), _ptr(out))
    return out


# ---- the solver (singleton in C; this class is a thin handle) ---------------

class Oracle:
    """Same call sequence as the product's C ABI, on host arrays.

    f arrays are numpy float64 of shape [Np, Ntheta] (row-major, theta fastest;
    PAPER.md L115).
    """

    def __init__(self, model: int, grid, domain, dt: float, threads: int = 1, **params):
        self.lib = _load()
        self.ntheta, self.np_ = int(grid[0]), int(grid[1])
        g = (ctypes.c_int * 2)(self.ntheta, self.np_)
        d = (ctypes.c_double * 4)(*[float(x) for x in domain])
        _check(self.lib.oracle_init(int(model), g, d, float(dt)), "init")
        self.lib.oracle_set_threads(int(threads))
        for k, v in params.items():
            key = {"eps": KEY_EPS, "bc_x": KEY_BC_X, "bc_p": KEY_BC_P, "spline": KEY_SPLINE, "order": KEY_ORDER}[k]
            _check(self.lib.oracle_set_param(key, float(v)), "set_param")

    @property
    def threads(self) -> int:
        return int(self.lib.oracle_get_threads())

    def upload(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64)
        assert f.shape == (self.np_, self.ntheta)
        _check(self.lib.oracle_upload(_ptr(f)), "upload")

    def download(self) -> np.ndarray:
        out = np.empty((self.np_, self.ntheta), dtype=np.float64)
        _check(self.lib.oracle_download(_ptr(out)), "download")
        return out

    def step(self, n: int = 1):
        _check(self.lib.oracle_step(int(n)), "step")

    def theta_sweep(self, tau: float):
        _check(self.lib.oracle_theta_sweep(float(tau)), "theta_sweep")

    def p_sweep(self, dt: float, force=None):
        if force is None:
            _check(self.lib.oracle_p_sweep(float(dt)), "p_sweep")
        else:
            F = np.ascontiguousarray(force, dtype=np.float64)
            assert F.shape == (self.ntheta,)
            _check(self.lib.oracle_p_sweep_with_force(_ptr(F), float(dt)), "p_sweep")

    def density(self) -> np.ndarray:
        out = np.empty(self.ntheta, dtype=np.float64)
        _check(self.lib.oracle_density(_ptr(out)), "density")
        return out

    def force(self) -> np.ndarray:
        out = np.empty(self.ntheta, dtype=np.float64)
        _check(self.lib.oracle_force(_ptr(out)), "force")
        return out

    def moments(self) -> np.ndarray:
        """{t, mass, P, K, U, Mx, My, E}"""
        out = np.empty(8, dtype=np.float64)
        _check(self.lib.oracle_moments(_ptr(out)), "moments")
        return out

    def casimirs(self) -> np.ndarray:
        """{S = -int f log f, C2 = int f^2, negative mass, max f}  (eq (18))"""
        out = np.empty(4, dtype=np.float64)
        _check(self.lib.oracle_casimirs(_ptr(out)), "casimirs")
        return out

    def close(self):
        self.lib.oracle_free()
