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
    ("cfg1", dict(ntheta=353, npts=61), dict()),                       # one-pass kernel, ragged row (plain stores)
    ("cfg1", dict(ntheta=352, npts=60), dict()),                       # one-pass kernel, bulk stores
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
