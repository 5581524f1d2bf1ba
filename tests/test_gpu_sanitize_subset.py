"""A small GPU subset that touches every kernel of the library on grids of a few thousand points: the cases
`compute-sanitizer` (memcheck, racecheck, initcheck) is run on (summaries in profiles/).
They are ordinary parity tests against the oracle and also run in the normal `-m gpu` suite."""
from __future__ import annotations

import math

import numpy as np
import pytest

from oracle import BC_PERIODIC, BC_ZERO, MODEL_HMF, MODEL_RING, MODEL_SHEET, MdOracle, Oracle, SPLINE_GS
from paper_1206_3229_b200 import binding as vb
from paper_1206_3229_b200 import inputs

pytestmark = pytest.mark.gpu
PI = math.pi


def rel_err(a, b):
    return float(np.max(np.abs(a - b))) / max(float(np.max(np.abs(b))), 1e-300)


@pytest.mark.parametrize("name,kw,params", [
    ("cfg1", dict(ntheta=353, npts=61), dict()),                       # one-pass step by the tile kernel (small grids)
    ("cfg1", dict(ntheta=353, npts=61), dict(tune_tile=2, tune_rc=2)), # warp-specialised one-pass kernel, ragged row (plain stores); ticketed density / force kernel
    ("cfg1", dict(ntheta=352, npts=60), dict(tune_tile=2)),            # warp-specialised one-pass kernel, bulk stores
    ("cfg1", dict(ntheta=352, npts=60), dict(precision=32)),           # fp32: difference form
    ("cfg1", dict(ntheta=128, npts=48), dict(fuse=1)),                 # theta x2 bulk kernel + p kernel
    ("cfg1", dict(ntheta=131, npts=40), dict(fuse=0)),                 # generic theta kernel
    ("cfg3", dict(ntheta=256, npts=48), dict()),                       # ring convolution
    ("cfg4", dict(ntheta=256, npts=64), dict()),                       # sheet: zero-extended x, prefix scan
    ("cfg1", dict(ntheta=96, npts=64), dict(spline=1)),                # global-spline kernels
    ("cfg1", dict(ntheta=128, npts=48), dict(order=4)),                # fourth-order composition
    ("cfg1", dict(ntheta=128, npts=48), dict(history=1)),              # per-step moments
])
def test_small_case_matches_oracle(name, kw, params):
    c = inputs.config(name, **kw)
    prec = params.get("precision", 64)
    op = {k: v for k, v in params.items() if k in ("order",)}
    if params.get("spline"):
        op["spline"] = SPLINE_GS
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=4, **op, **c["params"])
    o.upload(c["f0"])
    o.step(6)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], **params, **c["params"])
    g.upload(c["f0"])
    g.step(6)
    assert rel_err(g.download().astype(np.float64), o.download()) <= (1e-10 if prec == 64 else 1e-4)
    assert np.max(np.abs(g.moments() - o.moments())) <= (1e-10 if prec == 64 else 1e-4)
    cg, co = g.casimirs(), o.casimirs()
    assert np.allclose(cg, co, rtol=1e-4 if prec == 32 else 1e-9, atol=1e-9)
    g.close()
    o.close()


def test_small_md_matches_oracle():
    th, p = inputs.md_waterbag(3001, 1.0, 1.0)
    o = MdOracle(3001, 0.1)
    o.upload(th, p)
    o.step(5)
    g = vb.HmfMd(3001, 0.1)
    g.upload(th, p)
    g.step(5)
    a, b = g.download(), o.download()
    assert np.max(np.abs(a[0] - b[0])) < 1e-11 and np.max(np.abs(a[1] - b[1])) < 1e-11
    assert np.max(np.abs(g.moments() - o.moments())) < 1e-12
    g.close()
    o.close()


@pytest.mark.parametrize("name,kw,params", [
    ("cfg1", dict(ntheta=353, npts=61), dict()), ("cfg1", dict(ntheta=352, npts=60), dict(precision=32)),
    ("cfg1", dict(ntheta=353, npts=61), dict(tune_tile=2, tune_rc=2)), ("cfg5", dict(ntheta=1100, npts=640), dict(tune_tile=2)),
    ("cfg5", dict(ntheta=1100, npts=640), dict()), ("cfg3", dict(ntheta=256, npts=48), dict(fuse=1)),
    ("cfg4", dict(ntheta=256, npts=64), dict()), ("cfg1", dict(ntheta=96, npts=64), dict(spline=1)),
    ("cfg1", dict(ntheta=131, npts=40), dict(fuse=0, order=4)), ("cfg1", dict(ntheta=128, npts=48), dict(halo_lo=7, halo_hi=9, fuse=0)),
])
def test_no_byte_is_written_outside_the_attached_buffers(name, kw, params):
    """compute-sanitizer is closed on this pool (gpurun refuses it), so out-of-bounds WRITES are looked for directly:
    the state and work buffers handed to vlasov_attach sit between guard zones of 1 MiB filled with a pattern, every
    stage kind runs, and the guards must come back untouched (reads out of bounds would show up as parity failures
    of the tests above: the guards hold NaN patterns)."""
    import torch

    c = inputs.config(name, **kw)
    prec = params.get("precision", 64)
    vb.vlasov_init(c["model"], c["grid"], c["domain"], c["dt"])
    keys = {"precision": vb.KEY_PRECISION, "fuse": vb.KEY_FUSE, "spline": vb.KEY_SPLINE, "order": vb.KEY_ORDER,
            "halo_lo": vb.KEY_HALO_LO, "halo_hi": vb.KEY_HALO_HI, "tune_tile": vb.KEY_TUNE_TILE, "tune_rc": vb.KEY_TUNE_RC}
    for k, v in params.items():
        vb.vlasov_set_param(keys[k], v)
    for k, v in c["params"].items():
        vb.vlasov_set_param(vb.KEY_EPS, v)
    sb, wb, G = vb.vlasov_state_bytes(), vb.vlasov_workspace_bytes(), 1 << 20
    r = lambda b: (b + 255) & ~255
    buf = torch.full((G + r(sb) + G + r(wb) + G + 256,), 0xFF, dtype=torch.uint8, device="cuda")   # 0xFF..: NaN as fp64 / fp32
    base = (buf.data_ptr() + 255) & ~255
    o0 = base - buf.data_ptr()
    f_off, w_off = o0 + G, o0 + G + r(sb) + G
    buf[f_off:f_off + sb] = 0
    if params.get("halo_lo"):
        buf[w_off:w_off + wb] = 0   # a slab's halos are the caller's to fill (exchange): zeros here, not the NaN pattern
    vb.vlasov_attach(buf.data_ptr() + f_off, buf.data_ptr() + w_off, wb, torch.cuda.current_stream().cuda_stream)
    rows = c["grid"][1]
    f0 = c["f0"].astype(np.float64 if prec == 64 else np.float32)
    vb.vlasov_upload(np.ascontiguousarray(f0))
    vb.vlasov_sync()
    if params.get("halo_lo"):
        for st in (vb.SUB_THETA_HALF, vb.SUB_RHO, vb.SUB_FORCE_FROM_RHO, vb.SUB_P_FULL, vb.SUB_THETA_HALF):
            vb.vlasov_substep(st)
    else:
        vb.vlasov_step(5)
        vb.vlasov_step(1)
        for st in (vb.SUB_THETA_HALF, vb.SUB_THETA_TWICE, vb.SUB_FORCE, vb.SUB_P_FULL, vb.SUB_P_THETA_HALF, vb.SUB_P_THETA_TWICE):
            vb.vlasov_substep(st)
    vb.vlasov_moments()
    vb.vlasov_casimirs()
    out = np.empty((rows, c["grid"][0]), dtype=f0.dtype)
    vb.vlasov_download(out)
    assert np.all(np.isfinite(out))
    vb.vlasov_free()
    guards = [buf[:f_off], buf[f_off + sb:w_off], buf[w_off + wb:]]
    for gz in guards:
        assert bool((gz == 0xFF).all())
