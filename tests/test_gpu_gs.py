"""Parity of the GLOBAL SPLINE variant (VLASOV_KEY_SPLINE = 1, system (15))
of the CUDA path against the CPU oracle, element by element, through the C ABI.

The two sides share nothing: the oracle solves the cyclic tridiagonal system of every line (Thomas + Sherman-
Morrison) and evaluates eq (13); the CUDA kernels run the closed-form inverse as two first-order recursions.
Tolerances as for the FD path (north_star): fp64 max|df| <= 1e-10 max|f| after 100 steps, moments to 1e-10.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

from oracle import BC_PERIODIC, BC_ZERO, MODEL_FREE, MODEL_HMF, MODEL_RING, MODEL_SHEET, SPLINE_GS, Oracle
from paper_1206_3229_b200 import binding as vb
from paper_1206_3229_b200 import inputs

pytestmark = pytest.mark.gpu
PI = math.pi


def rel_err(a, b):
    den = float(np.max(np.abs(b)))
    return float(np.max(np.abs(a - b))) / (den if den > 0.0 else 1.0)


def rough_state(nt, npp, dom, seed=1):
    """smooth bump + 10 % white noise: the global spline couples every node of a line, noise exercises all of it"""
    rng = np.random.default_rng(seed)
    th = inputs.nodes(dom[0], dom[1], nt)
    p = inputs.nodes(dom[2], dom[3], npp)
    f = np.exp(-0.5 * (p[:, None] / 0.8) ** 2) * (1 + 0.4 * np.cos(th[None, :] - 0.3) + 0.1 * np.sin(3 * th[None, :]))
    return f + 0.1 * rng.random((npp, nt))


def pair(model, grid, dom, dt, f0, threads=8, precision=64, **params):
    o = Oracle(model, grid, dom, dt, threads=threads, spline=SPLINE_GS, **params)
    o.upload(f0)
    g = vb.Vlasov(model, grid, dom, dt, precision=precision, spline=vb.SPLINE_GS, **params)
    g.upload(f0)
    return o, g


GRIDS = [(64, 48), (279, 33), (1152, 37), (1153, 40), (2400, 32), (33, 32), (32, 300)]


@pytest.mark.parametrize("grid", GRIDS)
@pytest.mark.parametrize("bc_x", [BC_PERIODIC, BC_ZERO])
@pytest.mark.parametrize("dt", [0.1, -0.37, 9.0, 0.0])
def test_gs_theta_half_sweep(grid, bc_x, dt):
    dom = (-PI, PI, -4.0, 4.0)
    f0 = rough_state(grid[0], grid[1], dom)
    o, g = pair(MODEL_FREE, grid, dom, dt, f0, bc_x=bc_x)
    o.theta_sweep(0.5 * dt)
    g.substep(vb.SUB_THETA_HALF)
    assert rel_err(g.download(), o.download()) < 1e-13
    g.close()


@pytest.mark.parametrize("grid", [(64, 48), (130, 257), (33, 1000), (200, 32), (300, 41), (65, 520)])
@pytest.mark.parametrize("bc_p", [BC_ZERO, BC_PERIODIC])
@pytest.mark.parametrize("amp", [0.5, 30.0, 2000.0])
def test_gs_p_sweep_with_given_force(grid, bc_p, amp):
    dom = (-PI, PI, -4.0, 4.0)
    f0 = rough_state(grid[0], grid[1], dom, seed=3)
    th = inputs.nodes(dom[0], dom[1], grid[0])
    F = amp * np.sin(2 * th + 0.1) + 0.3 * amp
    o, g = pair(MODEL_FREE, grid, dom, 0.1, f0, bc_p=bc_p)
    o.p_sweep(0.1, force=F)
    g.set_force(F)
    g.substep(vb.SUB_P_FULL)
    assert rel_err(g.download(), o.download()) < 1e-13
    g.close()


@pytest.mark.parametrize("which,nhalf", [(vb.SUB_THETA_TWICE, 2), (vb.SUB_P_THETA_HALF, 1), (vb.SUB_P_THETA_TWICE, 2)])
def test_gs_composite_substeps(which, nhalf):
    """the composite test hooks run as separate passes with the global spline and leave density and force behind"""
    c = inputs.config("cfg1", ntheta=300, npts=200)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"])
    th = inputs.nodes(c["domain"][0], c["domain"][1], 300)
    F = 0.7 * np.sin(th + 0.2)
    if which != vb.SUB_THETA_TWICE:
        o.p_sweep(c["dt"], force=F)
        g.set_force(F)
    for _ in range(nhalf):
        o.theta_sweep(0.5 * c["dt"])
    g.substep(which)
    assert rel_err(g.download(), o.download()) < 1e-13
    if which != vb.SUB_THETA_TWICE:
        assert np.max(np.abs(g.force() - o.force())) <= 1e-12 * np.max(np.abs(o.force()))
    g.close()


def test_gs_integer_cell_shifts_are_exact_copies():
    """a = 0: w = (.., 0, 1, 0, ..) exactly, so the shifted line is a bit-exact copy (P2 holds for any f'')."""
    nt, npp = 128, 64
    dom = (0.0, float(nt), -4.0, 4.0)          # dx = 1; p_j tau integer for tau = 8: p_j = -4 + j/8
    f0 = rough_state(nt, npp, dom, seed=7)
    g = vb.Vlasov(MODEL_FREE, (nt, npp), dom, 16.0, spline=vb.SPLINE_GS)
    g.upload(f0)
    g.substep(vb.SUB_THETA_HALF)
    out = g.download()
    p = inputs.nodes(dom[2], dom[3], npp)
    for j in range(npp):
        assert np.array_equal(out[j], np.roll(f0[j], int(round(p[j] * 8.0))))
    g.close()


CASES = [
    ("cfg1", dict(), 100),                                   # HMF water-bag 256 x 256
    ("cfg1", dict(ntheta=300, npts=200), 60),                # ragged
    ("cfg2", dict(ntheta=512, npts=256), 100),               # HMF perturbed Gaussian
    ("cfg3", dict(ntheta=512, npts=256), 60),                # ring
    ("cfg4", dict(ntheta=512, npts=512), 100),               # sheet, zero-extended x
]


@pytest.mark.parametrize("name,kw,steps", CASES)
def test_gs_steps_match_the_oracle(name, kw, steps):
    c = inputs.config(name, **kw)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"])
    o.step(steps)
    g.step(steps)
    fo, fg = o.download(), g.download()
    assert rel_err(fg, fo) <= 1e-10
    assert np.max(np.abs(g.moments() - o.moments())) <= 1e-10
    g.close()


def test_gs_differs_from_fd_and_history_matches():
    """the variant really is another interpolation (not the FD path under another name), and the per-step
    records of vlasov_history agree with the oracle's moments step by step"""
    c = inputs.config("cfg1")
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=8, spline=SPLINE_GS)
    o.upload(c["f0"])
    gf = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"])
    gf.upload(c["f0"])
    gf.step(10)
    f_fd = gf.download()
    gf.close()
    g2 = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], spline=vb.SPLINE_GS, history=1)
    g2.upload(c["f0"])
    g2.step(10)
    hist = g2.history(10)
    f_gs = g2.download()
    g2.close()
    assert rel_err(f_gs, f_fd) > 1e-4
    for k in range(10):
        o.step(1)
        assert np.max(np.abs(hist[k] - o.moments())) <= 1e-10
    assert rel_err(f_gs, o.download()) <= 1e-11


def test_gs_fp32_storage():
    c = inputs.config("cfg1")
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], precision=32)
    o.step(100)
    g.step(100)
    assert rel_err(g.download().astype(np.float64), o.download()) <= 1e-4
    g.close()


def test_gs_refuses_short_axes():
    """vlasov_set_param itself refuses SPLINE = 1 on an axis shorter than 32 nodes (before anything is allocated), the
    context stays usable with the default spline, and a retry does not leak"""
    for grid in ((31, 64), (64, 8)):
        for _ in range(3):
            with pytest.raises(vb.VlasovError) as e:
                vb.Vlasov(MODEL_HMF, grid, (-PI, PI, -4.0, 4.0), 0.1, spline=vb.SPLINE_GS, attach=False)
            assert e.value.code == vb.EINVAL
        vb.vlasov_step(1)  # the context of the failed constructor is initialised and runs with the eq (16) spline
        vb.vlasov_free()


def test_gs_at_2048_first_steps_then_22_steps():
    """cfg 5 shape at 2048^2 (several chunks, bands and segments per axis): two steps element by element, then
    20 more on both sides: state and moments."""
    c = inputs.config("cfg5", ntheta=2048, npts=2048)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], threads=16)
    o.step(2)
    g.step(2)
    assert rel_err(g.download(), o.download()) <= 1e-12
    o.step(20)
    g.step(20)
    assert rel_err(g.download(), o.download()) <= 1e-11
    assert np.max(np.abs(g.moments() - o.moments())) <= 1e-11
    g.close()


# ----------------------------------------------------------------------------- full sizes of BASELINE.json's configs
def run_both_gs(c, steps):
    import os

    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=os.cpu_count() or 8, spline=SPLINE_GS, **c["params"])
    o.upload(c["f0"])
    o.step(steps)
    fo, mo = o.download(), o.moments()
    o.close()
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], spline=vb.SPLINE_GS, **c["params"])
    g.upload(c["f0"])
    g.step(steps)
    fg, mg = g.download(), g.moments()
    g.close()
    return fo, mo, fg, mg


@pytest.mark.parametrize("name,kw,steps", [("cfg2", {}, 100), ("cfg3", {}, 100), ("cfg4", {}, 100),
                                           ("cfg5", dict(n=4096), 40)])
def test_gs_full_size_steps_match_oracle(name, kw, steps):
    """cfg 2 (1024^2), cfg 3 (ring, 2048^2), cfg 4 (sheet, 4096^2, zero-extended x) for 100 steps and cfg 5 at 4096^2
    for 40, global spline on both sides, element by element (north_star: 1e-10 max|f|, moments 1e-10)."""
    c = inputs.config(name, **kw)
    fo, mo, fg, mg = run_both_gs(c, steps)
    assert rel_err(fg, fo) <= 1e-10
    assert np.max(np.abs(mg - mo)) <= 1e-10 * max(1.0, np.max(np.abs(mo)))


def test_gs_bench_size_20_steps_match_oracle():
    """8192^2 in the configuration bench.py --spline gs times: 20 steps element by element"""
    c = inputs.config("cfg5", n=8192)
    fo, mo, fg, mg = run_both_gs(c, 20)
    assert rel_err(fg, fo) <= 1e-10
    assert np.max(np.abs(mg - mo)) <= 1e-10 * max(1.0, np.max(np.abs(mo)))
