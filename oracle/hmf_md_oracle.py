"""ctypes front end of ``hmf_md_oracle.c`` (TEST INFRASTRUCTURE -- not part of the product).

The N-particle HMF molecular dynamics with the fourth-order symplectic integrator the paper used as its comparator
(Fig. 4, ref. [44]).  Only compiles the C file with gcc and marshals numpy
arrays; the arithmetic is in C.  Imports nothing from ``paper_1206_3229_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hmf_md_oracle.c")
_LIB = os.path.join(_HERE, "libhmf_md_oracle.so")
_lock = threading.Lock()
_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def build_md(force: bool = False) -> str:
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build_md())
            lib.oracle_md_init.argtypes = [ctypes.c_long, ctypes.c_double]
            lib.oracle_md_upload.argtypes = [_dp, _dp]
            lib.oracle_md_download.argtypes = [_dp, _dp]
            lib.oracle_md_step.argtypes = [ctypes.c_int]
            lib.oracle_md_moments.argtypes = [_dp]
            lib.oracle_md_potential_double_sum.restype = ctypes.c_double
            lib.oracle_md_free.restype = None
            _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError("%s failed with code %d" % (what, rc))


class MdOracle:
    """Singleton N-particle HMF integrator; theta, p are float64 arrays of length N."""

    def __init__(self, n: int, dt: float):
        self.n = int(n)
        _check(_load().oracle_md_init(self.n, float(dt)), "oracle_md_init")

    def upload(self, theta, p):
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        p = np.ascontiguousarray(p, dtype=np.float64)
        assert theta.shape == (self.n,) and p.shape == (self.n,)
        _check(_load().oracle_md_upload(theta.ctypes.data_as(_dp), p.ctypes.data_as(_dp)), "oracle_md_upload")

    def download(self):
        theta, p = np.empty(self.n), np.empty(self.n)
        _check(_load().oracle_md_download(theta.ctypes.data_as(_dp), p.ctypes.data_as(_dp)), "oracle_md_download")
        return theta, p

    def step(self, n: int = 1):
        _check(_load().oracle_md_step(int(n)), "oracle_md_step")

    def moments(self) -> np.ndarray:
        """{t, M_x, M_y, K/N, U/N, E/N, P/N, 0}"""
        out = np.empty(8)
        _check(_load().oracle_md_moments(out.ctypes.data_as(_dp)), "oracle_md_moments")
        return out

    def potential_double_sum(self) -> float:
        return float(_load().oracle_md_potential_double_sum())

    def close(self):
        _load().oracle_md_free()
