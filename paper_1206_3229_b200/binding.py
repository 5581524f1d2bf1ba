"""ctypes binding of ``csrc/libvlasov_b200.so`` (the C ABI of include/vlasov.h).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the ABI.  The module-level
functions carry the C names (``vlasov_init`` ...); ``Vlasov`` is a convenience handle that also owns the torch
tensors used as device memory (torch = device memory + stream, nothing else).

There is no CPU fallback: importing works without a GPU (so that the symbol table can be checked), but every
call that needs the device raises ``VlasovError`` if the library is missing or CUDA is unavailable.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

MODEL_FREE, MODEL_HMF, MODEL_RING, MODEL_SHEET = 0, 1, 2, 3
KEY_EPS, KEY_PRECISION, KEY_BC_X, KEY_BC_P, KEY_HISTORY, KEY_FUSE, KEY_PROFILE, KEY_SPLINE, KEY_ORDER, KEY_HALO_LO, KEY_HALO_HI = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11
SPLINE_FD, SPLINE_GS = 0, 1
KEY_TUNE_NW1, KEY_TUNE_NW2, KEY_TUNE_BANDS, KEY_TUNE_PSEG, KEY_TUNE_PTX, KEY_TUNE_GENERIC, KEY_TUNE_FBANDS, KEY_TUNE_FEDGE, KEY_TUNE_GRAPH, KEY_TUNE_PDL, KEY_TUNE_TILE, KEY_TUNE_RC, KEY_TUNE_HIST = 101, 102, 103, 104, 105, 106, 107, 108, 109, 110, 111, 112, 113
SUB_THETA_HALF, SUB_FORCE, SUB_P_FULL, SUB_THETA_TWICE, SUB_P_THETA_HALF, SUB_P_THETA_TWICE, SUB_RHO, SUB_FORCE_FROM_RHO = 0, 1, 2, 3, 4, 5, 6, 7
VEC_RHO, VEC_FORCE = 0, 1
OK, EINVAL, ENOTINIT, ECUDA, ENOMEM = 0, -1, -2, -3, -4

EXPORTS = (
    "vlasov_init", "vlasov_set_param", "vlasov_state_bytes", "vlasov_workspace_bytes", "vlasov_attach",
    "vlasov_state_ptr", "vlasov_upload", "vlasov_download", "vlasov_step", "vlasov_substep",
    "vlasov_get_vector", "vlasov_set_vector", "vlasov_vector_ptr", "vlasov_moments", "vlasov_casimirs", "vlasov_history", "vlasov_sync",
    "vlasov_launch_count", "vlasov_kernel_times", "vlasov_info", "vlasov_free", "vlasov_last_error",
)


MD_EXPORTS = (
    "hmf_md_init", "hmf_md_attach", "hmf_md_upload", "hmf_md_download", "hmf_md_step", "hmf_md_moments",
    "hmf_md_profile", "hmf_md_kernel_times", "hmf_md_launch_count", "hmf_md_free", "hmf_md_last_error",
)


# include/hmf_noalloc.h: the one entry point that allocates nothing
NOALLOC_EXPORTS = ("hmf_noalloc_moments", "hmf_noalloc_last_error")
NOALLOC_MAX_PARTICLES = 33554432


class VlasovError(RuntimeError):
    def __init__(self, code: int, what: str, msg: str):
        super().__init__("%s failed with code %d: %s" % (what, code, msg))
        self.code = code


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def library_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """dlopen the CUDA library (building it with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build_if_missing:
        try:
            path = _build.build_library()
        except Exception as exc:  # stale but present is still loadable; missing is fatal
            if not os.path.exists(path):
                raise VlasovError(ECUDA, "load", "CUDA library missing and nvcc build failed: %s" % exc)
    if not os.path.exists(path):
        raise VlasovError(ECUDA, "load", "%s not found (no CPU fallback exists)" % path)
    lib = ctypes.CDLL(path)
    vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    sig = {
        "vlasov_init": (ci, [ci, ctypes.POINTER(ci), _dp, cd]),
        "vlasov_set_param": (ci, [ci, cd]),
        "vlasov_state_bytes": (sz, []),
        "vlasov_workspace_bytes": (sz, []),
        "vlasov_attach": (ci, [vp, vp, sz, vp]),
        "vlasov_state_ptr": (ci, [ctypes.POINTER(vp)]),
        "vlasov_upload": (ci, [vp]),
        "vlasov_download": (ci, [vp]),
        "vlasov_step": (ci, [ci]),
        "vlasov_substep": (ci, [ci]),
        "vlasov_get_vector": (ci, [ci, _dp]),
        "vlasov_set_vector": (ci, [ci, _dp]),
        "vlasov_vector_ptr": (ci, [ci, ctypes.POINTER(vp)]),
        "vlasov_moments": (ci, [_dp]),
        "vlasov_casimirs": (ci, [_dp]),
        "vlasov_history": (ci, [_dp, ci]),
        "vlasov_sync": (ci, []),
        "vlasov_launch_count": (ci, [ctypes.POINTER(ctypes.c_ulonglong)]),
        "vlasov_info": (ci, [_dp, ci]),
        "vlasov_kernel_times": (ci, [_dp]),
        "vlasov_free": (None, []),
        "vlasov_last_error": (ctypes.c_char_p, []),
        # include/hmf_md.h
        "hmf_md_init": (ci, [ctypes.c_longlong, cd]),
        "hmf_md_attach": (ci, [vp, vp, vp]),
        "hmf_md_upload": (ci, [_dp, _dp]),
        "hmf_md_download": (ci, [_dp, _dp]),
        "hmf_md_step": (ci, [ci]),
        "hmf_md_moments": (ci, [_dp]),
        "hmf_md_profile": (ci, [ci]),
        "hmf_md_kernel_times": (ci, [_dp]),
        "hmf_md_launch_count": (ci, [ctypes.POINTER(ctypes.c_ulonglong)]),
        "hmf_md_free": (None, []),
        "hmf_md_last_error": (ctypes.c_char_p, []),
        # include/hmf_noalloc.h
        "hmf_noalloc_moments": (ci, [vp, vp, ctypes.c_longlong, cd, vp, vp]),
        "hmf_noalloc_last_error": (ctypes.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _chk(rc: int, what: str) -> int:
    if rc < 0:
        raise VlasovError(rc, what, (load().vlasov_last_error() or b"").decode())
    return rc


# ---- the C names ------------------------------------------------------------------------------------------

def vlasov_init(model: int, grid, domain, dt: float) -> None:
    g = (ctypes.c_int * 2)(int(grid[0]), int(grid[1]))
    d = (ctypes.c_double * 4)(*[float(x) for x in domain])
    _chk(load().vlasov_init(int(model), g, d, float(dt)), "vlasov_init")


def vlasov_set_param(key: int, value: float) -> None:
    _chk(load().vlasov_set_param(int(key), float(value)), "vlasov_set_param")


def vlasov_state_bytes() -> int:
    return int(load().vlasov_state_bytes())


def vlasov_workspace_bytes() -> int:
    return int(load().vlasov_workspace_bytes())


def vlasov_attach(f_dev_ptr: int, work_dev_ptr: int, work_bytes: int, cuda_stream: int) -> None:
    _chk(load().vlasov_attach(ctypes.c_void_p(f_dev_ptr), ctypes.c_void_p(work_dev_ptr), int(work_bytes),
                              ctypes.c_void_p(cuda_stream)), "vlasov_attach")


def vlasov_state_ptr() -> int:
    out = ctypes.c_void_p()
    _chk(load().vlasov_state_ptr(ctypes.byref(out)), "vlasov_state_ptr")
    return int(out.value or 0)


def vlasov_upload(f_host: np.ndarray) -> None:
    assert f_host.flags["C_CONTIGUOUS"]
    _chk(load().vlasov_upload(ctypes.c_void_p(f_host.ctypes.data)), "vlasov_upload")


def vlasov_upload_ptr(host_ptr: int) -> None:
    _chk(load().vlasov_upload(ctypes.c_void_p(host_ptr)), "vlasov_upload")


def vlasov_download(f_host: np.ndarray) -> None:
    assert f_host.flags["C_CONTIGUOUS"] and f_host.flags["WRITEABLE"]
    _chk(load().vlasov_download(ctypes.c_void_p(f_host.ctypes.data)), "vlasov_download")


def vlasov_download_ptr(host_ptr: int) -> None:
    _chk(load().vlasov_download(ctypes.c_void_p(host_ptr)), "vlasov_download")


def vlasov_step(n: int = 1) -> None:
    _chk(load().vlasov_step(int(n)), "vlasov_step")


def vlasov_substep(which: int) -> None:
    _chk(load().vlasov_substep(int(which)), "vlasov_substep")


def vlasov_get_vector(which: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _chk(load().vlasov_get_vector(int(which), out.ctypes.data_as(_dp)), "vlasov_get_vector")
    return out


def vlasov_set_vector(which: int, v) -> None:
    v = np.ascontiguousarray(v, dtype=np.float64)
    _chk(load().vlasov_set_vector(int(which), v.ctypes.data_as(_dp)), "vlasov_set_vector")


def vlasov_vector_ptr(which: int) -> int:
    out = ctypes.c_void_p()
    _chk(load().vlasov_vector_ptr(int(which), ctypes.byref(out)), "vlasov_vector_ptr")
    return int(out.value or 0)


def vlasov_moments() -> np.ndarray:
    out = np.empty(8, dtype=np.float64)
    _chk(load().vlasov_moments(out.ctypes.data_as(_dp)), "vlasov_moments")
    return out


def vlasov_casimirs() -> np.ndarray:
    out = np.empty(4, dtype=np.float64)
    _chk(load().vlasov_casimirs(out.ctypes.data_as(_dp)), "vlasov_casimirs")
    return out


def vlasov_history(max_steps: int) -> np.ndarray:
    out = np.empty((max(int(max_steps), 1), 8), dtype=np.float64)
    n = _chk(load().vlasov_history(out.ctypes.data_as(_dp), int(max_steps)), "vlasov_history")
    return out[:n]


def vlasov_sync() -> None:
    _chk(load().vlasov_sync(), "vlasov_sync")


def vlasov_launch_count() -> int:
    out = ctypes.c_ulonglong(0)
    _chk(load().vlasov_launch_count(ctypes.byref(out)), "vlasov_launch_count")
    return int(out.value)


def vlasov_kernel_times() -> dict:
    buf = np.zeros(12, dtype=np.float64)
    _chk(load().vlasov_kernel_times(buf.ctypes.data_as(_dp)), "vlasov_kernel_times")
    names = ["theta1", "theta2", "p", "force", "ptheta2", "ptheta1"]
    return {k: {"ms": float(buf[2 * i]), "launches": int(buf[2 * i + 1])} for i, k in enumerate(names)}


def vlasov_info() -> dict:
    buf = np.zeros(16, dtype=np.float64)
    n = _chk(load().vlasov_info(buf.ctypes.data_as(_dp), 16), "vlasov_info")
    names = ["sm_count", "theta2_ctas", "p_ctas", "theta2_bands", "theta2_warps", "theta1_warps", "theta1_ctas",
             "p_seg_len", "p_threads", "theta_bulk", "onepass", "onepass_ctas", "onepass_bands", "onepass_rows_per_band",
             "onepass_tile", "max_cluster"]
    return {k: int(buf[i]) for i, k in enumerate(names[:n])}


def vlasov_free() -> None:
    load().vlasov_free()


# ---- convenience handle -----------------------------------------------------------------------------------

class Vlasov:
    """Singleton solver handle.  ``f`` arrays are [Np, Ntheta], theta fastest.

    Device memory comes from torch (``torch.empty`` on ``cuda``) and is handed over with ``vlasov_attach``
    together with torch's current stream; nothing else of torch is used.
    """

    def __init__(self, model: int, grid, domain, dt: float, precision: int = 64, device: str = "cuda:0",
                 attach: bool = True, **params):
        import torch

        if not torch.cuda.is_available():
            raise VlasovError(ECUDA, "Vlasov", "no CUDA device: this library has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.ntheta, self.np_ = int(grid[0]), int(grid[1])
        self.dtype = np.float64 if precision == 64 else np.float32
        vlasov_init(model, grid, domain, dt)
        if precision != 64:
            vlasov_set_param(KEY_PRECISION, precision)
        keys = {"eps": KEY_EPS, "bc_x": KEY_BC_X, "bc_p": KEY_BC_P, "history": KEY_HISTORY, "fuse": KEY_FUSE, "profile": KEY_PROFILE, "spline": KEY_SPLINE, "order": KEY_ORDER, "halo_lo": KEY_HALO_LO, "halo_hi": KEY_HALO_HI,
                "tune_nw1": KEY_TUNE_NW1, "tune_nw2": KEY_TUNE_NW2, "tune_bands": KEY_TUNE_BANDS,
                "tune_pseg": KEY_TUNE_PSEG, "tune_ptx": KEY_TUNE_PTX, "tune_generic": KEY_TUNE_GENERIC,
                "tune_fbands": KEY_TUNE_FBANDS, "tune_fedge": KEY_TUNE_FEDGE, "tune_graph": KEY_TUNE_GRAPH, "tune_pdl": KEY_TUNE_PDL, "tune_tile": KEY_TUNE_TILE, "tune_rc": KEY_TUNE_RC, "tune_hist": KEY_TUNE_HIST}
        for k, v in params.items():
            vlasov_set_param(keys[k], float(v))
        self.f_dev = self.work_dev = None
        if attach:
            tdt = torch.float64 if precision == 64 else torch.float32
            # rows of a state buffer: the grid's, plus the halos of a slab (VLASOV_KEY_HALO_LO / _HI)
            self.rows_ext = vlasov_state_bytes() // (self.ntheta * (8 if precision == 64 else 4))
            self.f_dev = torch.zeros((self.rows_ext, self.ntheta), dtype=tdt, device=self.device)
            self.work_dev = torch.empty(vlasov_workspace_bytes() + 256, dtype=torch.uint8, device=self.device)
            wp = (self.work_dev.data_ptr() + 255) & ~255
            self.stream = torch.cuda.current_stream(self.device)
            vlasov_attach(self.f_dev.data_ptr(), wp, vlasov_workspace_bytes(), self.stream.cuda_stream)
            off = wp - self.work_dev.data_ptr()
            self.f_alt = self.work_dev[off:off + self.f_dev.numel() * self.f_dev.element_size()].view(tdt).view(
                self.rows_ext, self.ntheta)  # the second state buffer (the passes ping-pong between the two)

    def current_state_tensor(self):
        """torch view [rows (+ halos), Ntheta] of the buffer that holds f now (attached buffers only)"""
        ptr = vlasov_state_ptr()
        if ptr == self.f_dev.data_ptr():
            return self.f_dev
        assert ptr == self.f_alt.data_ptr()
        return self.f_alt

    def upload(self, f) -> None:
        f = np.ascontiguousarray(f, dtype=self.dtype)
        assert f.shape == (self.np_, self.ntheta)
        vlasov_upload(f)
        vlasov_sync()  # f may be a temporary: do not let it die under the asynchronous copy

    def download(self) -> np.ndarray:
        out = np.empty((self.np_, self.ntheta), dtype=self.dtype)
        vlasov_download(out)
        return out

    def step(self, n: int = 1) -> None:
        vlasov_step(n)

    def substep(self, which: int) -> None:
        vlasov_substep(which)

    def density(self) -> np.ndarray:
        return vlasov_get_vector(VEC_RHO, self.ntheta)

    def force(self) -> np.ndarray:
        return vlasov_get_vector(VEC_FORCE, self.ntheta)

    def set_force(self, F) -> None:
        vlasov_set_vector(VEC_FORCE, F)

    def moments(self) -> np.ndarray:
        return vlasov_moments()

    def history(self, n: int) -> np.ndarray:
        return vlasov_history(n)

    def sync(self) -> None:
        vlasov_sync()

    def casimirs(self) -> np.ndarray:
        """{S = -int f log f, C2 = int f^2, negative mass, max f}  (eq (18))"""
        return vlasov_casimirs()

    def info(self) -> dict:
        return vlasov_info()

    def close(self) -> None:
        vlasov_free()
        self.f_dev = self.work_dev = None


# ---- HMF molecular dynamics (include/hmf_md.h) -------------------------------------------------------------

def _chk_md(rc: int, what: str) -> int:
    if rc < 0:
        raise VlasovError(rc, what, (load().hmf_md_last_error() or b"").decode())
    return rc


def hmf_md_launch_count() -> int:
    out = ctypes.c_ulonglong(0)
    _chk_md(load().hmf_md_launch_count(ctypes.byref(out)), "hmf_md_launch_count")
    return int(out.value)


def hmf_noalloc_moments(theta_ptr: int, p_ptr: int, n: int, t: float, out_ptr: int, stream: int = 0) -> None:
    """include/hmf_noalloc.h: the moments of n particles (device pointers of the caller, out_ptr: 8 doubles on the device),
    enqueued on `stream` (a cudaStream_t as an integer); calls no cudaMalloc.  Argument marshalling only."""
    rc = load().hmf_noalloc_moments(ctypes.c_void_p(theta_ptr), ctypes.c_void_p(p_ptr), int(n), float(t),
                                    ctypes.c_void_p(out_ptr), ctypes.c_void_p(stream))
    if rc < 0:
        raise VlasovError(rc, "hmf_noalloc_moments", (load().hmf_noalloc_last_error() or b"").decode())


class HmfMd:
    """N-particle HMF molecular dynamics (eqs (7)-(8), L206): argument marshalling only.  theta, p are
    float64 arrays of length N; torch supplies the device memory and the stream."""

    def __init__(self, n: int, dt: float, device: str = "cuda:0", attach: bool = True):
        import torch

        if not torch.cuda.is_available():
            raise VlasovError(ECUDA, "HmfMd", "no CUDA device: this library has no CPU fallback")
        self.n = int(n)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        _chk_md(load().hmf_md_init(self.n, float(dt)), "hmf_md_init")
        self.theta_dev = self.p_dev = None
        if attach:
            self.theta_dev = torch.zeros(self.n, dtype=torch.float64, device=self.device)
            self.p_dev = torch.zeros(self.n, dtype=torch.float64, device=self.device)
            stream = torch.cuda.current_stream(self.device).cuda_stream
            _chk_md(load().hmf_md_attach(ctypes.c_void_p(self.theta_dev.data_ptr()), ctypes.c_void_p(self.p_dev.data_ptr()),
                                         ctypes.c_void_p(stream)), "hmf_md_attach")

    def upload(self, theta, p) -> None:
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        p = np.ascontiguousarray(p, dtype=np.float64)
        assert theta.shape == (self.n,) and p.shape == (self.n,)
        _chk_md(load().hmf_md_upload(theta.ctypes.data_as(_dp), p.ctypes.data_as(_dp)), "hmf_md_upload")
        self.moments()  # blocks: theta, p may be temporaries

    def upload_ptr(self, theta_ptr: int, p_ptr: int) -> None:
        _chk_md(load().hmf_md_upload(ctypes.cast(theta_ptr, _dp), ctypes.cast(p_ptr, _dp)), "hmf_md_upload")

    def download_ptr(self, theta_ptr: int, p_ptr: int) -> None:
        _chk_md(load().hmf_md_download(ctypes.cast(theta_ptr, _dp), ctypes.cast(p_ptr, _dp)), "hmf_md_download")

    def download(self):
        theta, p = np.empty(self.n), np.empty(self.n)
        _chk_md(load().hmf_md_download(theta.ctypes.data_as(_dp), p.ctypes.data_as(_dp)), "hmf_md_download")
        return theta, p

    def step(self, n: int = 1) -> None:
        _chk_md(load().hmf_md_step(int(n)), "hmf_md_step")

    def moments(self) -> np.ndarray:
        """{t, M_x, M_y, K/N, U/N, E/N, P/N, 0}"""
        out = np.empty(8)
        _chk_md(load().hmf_md_moments(out.ctypes.data_as(_dp)), "hmf_md_moments")
        return out

    def profile(self, on: bool) -> None:
        _chk_md(load().hmf_md_profile(int(on)), "hmf_md_profile")

    def kernel_times(self):
        out = np.zeros(2)
        _chk_md(load().hmf_md_kernel_times(out.ctypes.data_as(_dp)), "hmf_md_kernel_times")
        return float(out[0]), int(out[1])

    def close(self) -> None:
        load().hmf_md_free()
        self.theta_dev = self.p_dev = None
