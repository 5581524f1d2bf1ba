"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (north_star): fp64 max|df| <= 1e-10 max|f| after 100 steps, moments to 1e-10.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

from oracle import BC_PERIODIC, BC_ZERO, MODEL_FREE, MODEL_HMF, MODEL_RING, MODEL_SHEET, Oracle
from paper_1206_3229_b200 import binding as vb
from paper_1206_3229_b200 import inputs

pytestmark = pytest.mark.gpu
PI = math.pi
TOL = 1e-10


def rel_err(a, b):
    den = float(np.max(np.abs(b)))
    return float(np.max(np.abs(a - b))) / (den if den > 0.0 else 1.0)


def smooth_state(nt, npp, dom, seed=1):
    rng = np.random.default_rng(seed)
    th = inputs.nodes(dom[0], dom[1], nt)
    p = inputs.nodes(dom[2], dom[3], npp)
    f = np.exp(-0.5 * (p[:, None] / 0.8) ** 2) * (1 + 0.4 * np.cos(th[None, :] - 0.3) + 0.1 * np.sin(3 * th[None, :]))
    return f + 1e-3 * rng.random((npp, nt))


def pair(model, grid, dom, dt, f0, threads=8, gpu_params=None, **params):
    o = Oracle(model, grid, dom, dt, threads=threads, **params)
    o.upload(f0)
    g = vb.Vlasov(model, grid, dom, dt, **params, **(gpu_params or {}))
    g.upload(f0)
    return o, g


# ----------------------------------------------------------------------------- single stages (T1)
GRIDS = [(64, 48), (279, 33), (280, 65), (1000, 37), (2233, 20), (31, 9), (1, 5), (7, 1)]


@pytest.mark.parametrize("grid", GRIDS)
@pytest.mark.parametrize("bc_x", [BC_PERIODIC, BC_ZERO])
@pytest.mark.parametrize("dt", [0.1, -0.37, 9.0, 0.0])
def test_theta_half_sweep(grid, bc_x, dt):
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom)
    o, g = pair(MODEL_FREE, grid, dom, dt, f0, bc_x=bc_x)
    o.theta_sweep(0.5 * dt)
    g.substep(vb.SUB_THETA_HALF)
    assert rel_err(g.download(), o.download()) < 1e-13
    g.close()


@pytest.mark.parametrize("grid", GRIDS)
@pytest.mark.parametrize("bc_x", [BC_PERIODIC, BC_ZERO])
@pytest.mark.parametrize("dt", [0.1, -0.37, 9.0])
def test_theta_twice_fused_equals_two_oracle_half_sweeps(grid, bc_x, dt):
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom, seed=2)
    o, g = pair(MODEL_FREE, grid, dom, dt, f0, bc_x=bc_x)
    o.theta_sweep(0.5 * dt)
    o.theta_sweep(0.5 * dt)
    g.substep(vb.SUB_THETA_TWICE)
    assert rel_err(g.download(), o.download()) < 1e-13
    g.close()


@pytest.mark.parametrize("grid", [(64, 48), (130, 257), (33, 1000), (200, 10), (5, 3), (300, 41)])
@pytest.mark.parametrize("bc_p", [BC_ZERO, BC_PERIODIC])
@pytest.mark.parametrize("amp", [0.5, 30.0, 2000.0])
def test_p_sweep_with_given_force(grid, bc_p, amp):
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom, seed=3)
    th = inputs.nodes(dom[0], dom[1], grid[0])
    F = amp * np.sin(2 * th + 0.1) + 0.3 * amp
    o, g = pair(MODEL_FREE, grid, dom, 0.1, f0, bc_p=bc_p)
    o.p_sweep(0.1, force=F)
    g.set_force(F)
    g.substep(vb.SUB_P_FULL)
    assert rel_err(g.download(), o.download()) < 1e-13
    g.close()


@pytest.mark.parametrize("model,dom", [(MODEL_HMF, (-PI, PI, -4.0, 4.0)), (MODEL_RING, (-PI, PI, -3.0, 3.0)),
                                       (MODEL_SHEET, (-10.0, 10.0, -4.0, 4.0)), (MODEL_FREE, (-PI, PI, -4.0, 4.0))])
@pytest.mark.parametrize("grid", [(64, 48), (300, 129), (1024, 70), (1500, 40), (2048, 64)])
@pytest.mark.parametrize("rc", [0, 2])
def test_density_force_and_moments(model, dom, grid, rc):
    """rc = 0: HMF on theta axes of up to 1024 columns takes the thread-block-cluster kernel (rho_force_cluster_kernel),
    rc = 2 (TUNE_RC): the ticketed rho_force_kernel that every other grid and model takes."""
    f0 = smooth_state(grid[0], grid[1], dom, seed=4)
    o, g = pair(model, grid, dom, 0.05, f0, gpu_params=dict(tune_rc=rc))
    g.substep(vb.SUB_FORCE)
    rho_o, F_o = o.density(), o.force()
    assert np.max(np.abs(g.density() - rho_o)) <= 1e-13 * np.max(np.abs(rho_o))
    assert np.max(np.abs(g.force() - F_o)) <= 1e-12 * max(np.max(np.abs(F_o)), 1e-300)
    mo, mg = o.moments(), g.moments()
    assert np.max(np.abs(mg - mo)) <= 1e-12 * np.max(np.abs(mo))
    g.close()


def test_density_after_theta_sweep_epilogue():
    """The column sums the theta kernel leaves behind feed the force of the step (eq (10) uses f_I)."""
    c = inputs.config("cfg1", ntheta=300, npts=200)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"])
    o.theta_sweep(0.5 * c["dt"])
    F_o = o.force()
    g.step(1)
    assert np.max(np.abs(g.force() - F_o)) <= 1e-12 * np.max(np.abs(F_o))
    assert np.max(np.abs(g.density() - o.density())) <= 1e-13 * np.max(o.density())
    g.close()


# ----------------------------------------------------------------------------- one-pass kernel (p + theta)
ONEPASS_GRIDS = [(64, 48), (352, 30), (353, 61), (1000, 137), (2233, 25), (31, 9), (1, 5), (7, 1), (720, 700), (1023, 1001)]


@pytest.mark.parametrize("grid", ONEPASS_GRIDS)
@pytest.mark.parametrize("bc_p", [BC_ZERO, BC_PERIODIC])
@pytest.mark.parametrize("which,dt,amp", [(1, 0.1, 0.5), (2, 0.1, 0.5), (2, -0.37, 30.0), (1, 9.0, 2000.0),
                                          (2, 9.0, 30.0), (2, 3.0, 0.0), (2, 0.1, 300.0), (1, 0.1, 7.0)])
@pytest.mark.parametrize("tile", [1, 2])
def test_one_pass_p_then_theta(grid, bc_p, which, dt, amp, tile):
    """p shift with a given force, then one or two half theta shifts, then density and force of the result:
    the one-pass kernel against the oracle's separate sweeps (eqs (11), (12), (9), (10)).  tile = 1: the tile kernel of
    small grids (strang_tile_kernel), tile = 2: the warp-specialised kernel of the large ones on the same small grid."""
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom, seed=5)
    th = inputs.nodes(dom[0], dom[1], grid[0])
    F = amp * np.sin(2 * th + 0.1) + 0.3 * amp
    o, g = pair(MODEL_HMF, grid, dom, dt, f0, bc_p=bc_p, gpu_params=dict(tune_tile=tile))
    o.p_sweep(dt, force=F)
    for _ in range(which):
        o.theta_sweep(0.5 * dt)
    g.set_force(F)
    # which path runs is part of the contract of every case: forward steps whose row shifts stay within one turn of the
    # circle take the one-pass kernel; a backward step (the row shifts grow with p) or a shift of several turns (dt = 9)
    # takes the separate kernels, unless one axis has a single node (then all row shifts are equal)
    expect_onepass = int(0.0 < dt <= 3.0 or min(grid) == 1)
    assert g.info()["onepass"] == expect_onepass
    # ... and which of the two one-pass kernels: the tile kernel wherever the one-pass path applies and the row shift
    # drifts by less than a column block inside 16 rows
    if dt != 3.0:  # (at dt = 3 the row shift drifts by more than a column block inside 16 rows on some of the grids)
        assert g.info()["onepass_tile"] == int(tile == 1 and expect_onepass == 1)
    else:
        assert g.info()["onepass_tile"] <= int(tile == 1)
    g.substep(vb.SUB_P_THETA_TWICE if which == 2 else vb.SUB_P_THETA_HALF)
    fo = o.download()
    assert rel_err(g.download(), fo) < 1e-13
    rho_o = o.density()
    assert np.max(np.abs(g.density() - rho_o)) <= 1e-13 * np.max(np.abs(rho_o))
    F_o = o.force()
    assert np.max(np.abs(g.force() - F_o)) <= 1e-12 * max(np.max(np.abs(F_o)), np.max(np.abs(rho_o)))
    g.close()


@pytest.mark.parametrize("grid", ONEPASS_GRIDS + [(4096, 40)])
@pytest.mark.parametrize("bc_p", [BC_ZERO, BC_PERIODIC])
@pytest.mark.parametrize("which,dt,amp", [(1, 0.1, 0.5), (2, 0.1, 0.5), (2, 0.45, 30.0), (2, 2.5, 3.0), (1, 9.0, 2000.0), (2, 3.0, 0.0)])
def test_one_pass_zero_extended_theta_axis(grid, bc_p, which, dt, amp):
    """the same with a zero-extended theta axis (the sheet model, BASELINE.json cfg 4): source columns beyond the ends are
    zeros, outputs beyond them are dropped, and near the ends the two half shifts are applied one after the other because
    the first is cropped to the grid before the second reads it (noise on every node, so the crop matters)"""
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom, seed=8) + 0.3
    th = inputs.nodes(dom[0], dom[1], grid[0])
    F = amp * np.sin(2 * th + 0.1) + 0.3 * amp
    o, g = pair(MODEL_SHEET, grid, dom, dt, f0, bc_p=bc_p)
    o.p_sweep(dt, force=F)
    for _ in range(which):
        o.theta_sweep(0.5 * dt)
    g.set_force(F)
    # the path is asserted in every case: a shift range of more than four domain lengths (dt = 9) takes the separate
    # kernels, everything else the one-pass kernel
    assert g.info()["onepass"] == int(dt <= 3.0)
    g.substep(vb.SUB_P_THETA_TWICE if which == 2 else vb.SUB_P_THETA_HALF)
    fo = o.download()
    assert rel_err(g.download(), fo) < 1e-13
    rho_o = o.density()
    assert np.max(np.abs(g.density() - rho_o)) <= 1e-13 * np.max(np.abs(rho_o))
    g.close()


@pytest.mark.parametrize("fbands", [1, 3, 50])
def test_one_pass_band_split_does_not_change_the_result(fbands):
    dom = (-PI, PI, -4.0, 4.0)
    grid = (800, 300)
    f0 = smooth_state(grid[0], grid[1], dom, seed=6)
    th = inputs.nodes(dom[0], dom[1], grid[0])
    F = 3.0 * np.sin(th + 0.2)
    o, g = pair(MODEL_HMF, grid, dom, 0.7, f0, gpu_params=dict(tune_fbands=fbands, tune_tile=2))
    o.p_sweep(0.7, force=F)
    o.theta_sweep(0.35)
    o.theta_sweep(0.35)
    g.set_force(F)
    g.substep(vb.SUB_P_THETA_TWICE)
    assert rel_err(g.download(), o.download()) < 1e-13
    assert np.max(np.abs(g.density() - o.density())) <= 1e-13 * np.max(o.density())
    g.close()


# ----------------------------------------------------------------------------- full steps (T2, T3)
CASES = [
    ("cfg1", dict()),                        # the real cfg 1: 256 x 256, 100 steps
    ("cfg2", dict(ntheta=256, npts=320)),
    ("cfg3", dict(ntheta=320, npts=256)),
    ("cfg4", dict(ntheta=512, npts=300)),
    ("cfg5", dict(ntheta=600, npts=280)),
]


@pytest.mark.parametrize("name,kw", CASES)
@pytest.mark.parametrize("fuse", [2, 1, 0])
def test_100_steps_match_oracle(name, kw, fuse):
    c = inputs.config(name, **kw)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], gpu_params=dict(fuse=fuse), **c["params"])
    o.step(100)
    g.step(100)
    fo, fg = o.download(), g.download()
    assert rel_err(fg, fo) <= TOL
    mo, mg = o.moments(), g.moments()
    assert np.max(np.abs(mg - mo)) <= TOL * max(1.0, np.max(np.abs(mo)))
    assert mg[0] == pytest.approx(100 * c["dt"])
    g.close()


@pytest.mark.parametrize("name,kw", [c for c in CASES if c[0] != "cfg4"])
def test_100_steps_match_oracle_large_grid_kernel_on_small_grids(name, kw):
    _run_100_steps_large_grid_kernels(name, kw)


def _run_100_steps_large_grid_kernels(name, kw):
    """The default one-pass path of these grids is the tile kernel (test above, fuse = 2); the warp-specialised kernel that
    the large grids take is held to the same bar on them (TUNE_TILE = 2), and so is their density / force kernel (TUNE_RC = 2:
    the ticketed kernel instead of the thread-block cluster).  (cfg 4 has a zero-extended x axis: always the warp-specialised
    kernel.)"""
    c = inputs.config(name, **kw)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], gpu_params=dict(fuse=2, tune_tile=2, tune_rc=2), **c["params"])
    assert g.info()["onepass"] == 1 and g.info()["onepass_tile"] == 0
    o.step(100)
    g.step(100)
    assert rel_err(g.download(), o.download()) <= TOL
    mo, mg = o.moments(), g.moments()
    assert np.max(np.abs(mg - mo)) <= TOL * max(1.0, np.max(np.abs(mo)))
    g.close()


@pytest.mark.parametrize("grid", [(256, 256), (1000, 137), (353, 61), (2048, 96), (1024, 960)])  # the three tile shapes
@pytest.mark.parametrize("bc_p", [BC_ZERO, BC_PERIODIC])
@pytest.mark.parametrize("which", [1, 2])
@pytest.mark.parametrize("precision", [64, 32])
def test_tile_kernel_and_large_grid_kernel_agree_bit_for_bit(grid, bc_p, which, precision):
    """Both one-pass kernels apply the same sequence of floating-point operations to every grid point (ten FMAs of the
    momentum shift, 10 or 19 of the theta weights; fp32: the same difference form): with the same force, f after the pass
    is the same bits; the density differs only in the order of its column sums."""
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom, seed=11)
    th = inputs.nodes(dom[0], dom[1], grid[0])
    F = 0.8 * np.sin(th + 0.3) + 0.1
    outs, rhos = [], []
    for tile in (1, 2):
        g = vb.Vlasov(MODEL_HMF, grid, dom, 0.1, bc_p=bc_p, tune_tile=tile, precision=precision)
        g.upload(f0.astype(np.float32) if precision == 32 else f0)
        assert g.info()["onepass"] == 1 and g.info()["onepass_tile"] == (1 if tile == 1 else 0)
        g.set_force(F)
        g.substep(vb.SUB_P_THETA_TWICE if which == 2 else vb.SUB_P_THETA_HALF)
        outs.append(g.download())
        rhos.append(g.density())
        g.close()
    assert np.array_equal(outs[0], outs[1])
    assert np.max(np.abs(rhos[0] - rhos[1])) <= 1e-13 * np.max(np.abs(rhos[1]))


@pytest.mark.parametrize("name,kw", [("cfg1", dict(n=128)), ("cfg1", dict()), ("cfg2", dict(ntheta=320, npts=256)),
                                     ("cfg5", dict(ntheta=700, npts=260)), ("cfg3", dict(ntheta=320, npts=256))])
@pytest.mark.parametrize("hist,tile", [(0, 0), (0, 2), (2, 0)])
def test_history_records_every_step_and_matches_oracle(name, kw, hist, tile):
    """HISTORY = 1: the eight moments after EVERY step against the oracle's.  hist = 0: with the HMF model the history comes off
    the one-pass path (per-row sums of the stored, half-shifted state and the row's Fourier factor, history_rows_kernel; the
    sums from the tile kernel itself on small grids, tile = 0, from a read pass behind the warp-specialised kernel of the large
    grids, tile = 2); hist = 2 (TUNE_HIST) and the ring model: the separate passes with a moments read pass per step."""
    c = inputs.config(name, **kw)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"],
                gpu_params=dict(history=1, tune_hist=hist, tune_tile=tile), **c["params"])
    g.step(20)
    h = g.history(20)
    assert h.shape == (20, 8)
    for k in range(20):
        o.step(1)
        mo = o.moments()
        assert np.max(np.abs(h[k] - mo)) <= TOL * max(1.0, np.max(np.abs(mo))), k
    assert rel_err(g.download(), o.download()) <= TOL
    g.step(3)  # a second call: the history restarts, the clock does not
    o.step(3)
    h = g.history(3)
    assert abs(h[2][0] - 23 * c["dt"]) < 1e-12 and np.max(np.abs(h[2] - o.moments())) <= TOL * max(1.0, np.max(np.abs(o.moments())))
    g.close()


@pytest.mark.parametrize("fuse", [2, 1])
def test_fused_multi_step_equals_single_steps(fuse):
    """P18: step(5) == 5 x step(1).  FUSE = 1 keeps the operation order (the intermediate row is rounded to fp64
    in both): bitwise.  FUSE = 2 applies two half shifts with the composite weights W = w * w: round-off."""
    c = inputs.config("cfg5", ntheta=700, npts=260)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], fuse=fuse)
    g.upload(c["f0"])
    g.step(5)
    a = g.download()
    g.close()
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], fuse=fuse)
    g.upload(c["f0"])
    for _ in range(5):
        g.step(1)
    b = g.download()
    g.close()
    if fuse == 1:
        assert np.array_equal(a, b)
    else:
        assert rel_err(a, b) < 1e-13


@pytest.mark.parametrize("tile", [1, 2])
def test_one_pass_is_reproducible_run_to_run(tile):
    """The density partials are accumulated with atomic adds of at most two terms per entry: same bits every run."""
    c = inputs.config("cfg5", ntheta=1500, npts=900)
    outs = []
    for _ in range(3):
        g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], tune_tile=tile)
        g.upload(c["f0"])
        g.step(7)
        outs.append(g.download())
        g.close()
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])


@pytest.mark.parametrize("name,kw,steps", [("cfg1", dict(), 40), ("cfg2", dict(n=256), 0), ("cfg3", dict(ntheta=320, npts=256), 25),
                                           ("cfg4", dict(ntheta=512, npts=300), 25), ("cfg5", dict(ntheta=1500, npts=700), 10)])
def test_casimirs_match_oracle(name, kw, steps):
    """Entropy, int f^2, negative mass and max f of eq (18) (L183-L188) of the evolved state: CUDA reduction against
    the oracle's long-double sums (1e-12 relative: one ulp of log per node, different summation order)."""
    c = inputs.config(name, **kw)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], **c["params"])
    if steps:
        o.step(steps)
        g.step(steps)
    co, cg = o.casimirs(), g.casimirs()
    scale = np.array([abs(co[0]), co[1], max(abs(co[2]), 1e-3 * co[1]), abs(co[3])])
    assert np.all(np.abs(cg - co) <= 1e-10 * np.maximum(scale, 1e-300)), (co, cg)
    if steps:
        assert co[2] < 0.0 or name == "cfg2"  # the water-bags undershoot at their edges: negative mass is real
    g.close()


def test_papers_sheet_run_periodic_boundaries_energy_error_and_entropy():
    """The paper's own sheet set-up (L145-L150: x, p in [-2, 2], periodic in both, water-bag x0 = 1, p0 = 0.5 with its
    edges, dt = 0.1; Table 2, Fig. 2): the CUDA path (one-pass kernel: x is periodic) against the
    oracle after 300 steps, the energy error inside Table 2's range, the norm to round-off, the entropy rising."""
    n = 512
    dom = (-2.0, 2.0, -2.0, 2.0)
    x = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = np.where((np.abs(x)[None, :] <= 1.0) & (np.abs(p)[:, None] <= 0.5), 0.5, 0.0)
    o, g = pair(MODEL_SHEET, (n, n), dom, 0.1, f0, bc_x=BC_PERIODIC, bc_p=BC_PERIODIC)
    assert g.info()["onepass"] == 1
    m0, c0 = g.moments(), g.casimirs()
    de = dn = 0.0
    for _ in range(30):
        g.step(10)
        m = g.moments()
        de = max(de, abs(m[7] - m0[7]) / abs(m0[7]))
        dn = max(dn, abs(m[1] - m0[1]) / m0[1])
    o.step(300)
    assert rel_err(g.download(), o.download()) <= TOL
    assert np.max(np.abs(g.moments() - o.moments())) <= TOL
    assert np.allclose(g.casimirs(), o.casimirs(), rtol=1e-10, atol=1e-13)
    assert 1e-5 <= de <= 1e-3       # Table 2: 4e-4 at n = 512 (run length not stated)
    assert dn <= 1e-12              # exact telescoping (the paper reports 2e-7, D14)
    assert g.casimirs()[0] > c0[0]  # Fig. 2
    g.close()


def test_casimirs_fp32_state():
    c = inputs.config("cfg5", ntheta=640, npts=320)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], precision=32)
    f32 = c["f0"].astype(np.float32)
    g.upload(f32)
    cg = g.casimirs()
    g.close()
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=8)
    o.upload(f32.astype(np.float64))
    co = o.casimirs()
    o.close()
    assert np.allclose(cg, co, rtol=1e-12, atol=0)


def test_graph_launches_change_nothing():
    """Steady-state step pairs launched as CUDA graphs (default) and as plain launches: same kernels, same bits."""
    c = inputs.config("cfg5", ntheta=900, npts=500)
    outs, launches = [], []
    for graph in (1, 0):
        g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], tune_graph=graph)
        g.upload(c["f0"])
        l0 = vb.vlasov_launch_count()
        g.step(9)
        g.step(4)
        outs.append(g.download())
        launches.append(vb.vlasov_launch_count() - l0)
        g.close()
    assert np.array_equal(outs[0], outs[1])
    assert launches[0] == launches[1] == (1 + 2 * 9) + (1 + 2 * 4)


def test_non_blocking_stream_can_be_attached():
    """Every torch.cuda.Stream() is a non-blocking stream: nothing orders it after the legacy default stream on which
    vlasov_init's tables are uploaded and its counters zeroed; the library synchronises once before the first launch."""
    import torch

    c = inputs.config("cfg5", ntheta=1100, npts=640)
    outs = []
    for own_stream in (False, True):
        s = torch.cuda.Stream() if own_stream else torch.cuda.current_stream()
        with torch.cuda.stream(s):
            g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"])
            g.upload(c["f0"])
            g.step(6)
            outs.append((g.download(), g.moments()))
            g.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_library_owned_buffers_and_checkpoint_roundtrip():
    c = inputs.config("cfg1", n=96)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], attach=False)
    g.upload(c["f0"])
    assert np.array_equal(g.download(), c["f0"])
    g.step(3)
    ck = g.download()
    g.step(2)
    ref = g.download()
    g.close()
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"])
    g.upload(ck)
    g.step(2)
    assert np.array_equal(g.download(), ref)
    g.close()


def test_errors():
    with pytest.raises(vb.VlasovError):
        vb.vlasov_init(9, (8, 8), (-1, 1, -1, 1), 0.1)
    with pytest.raises(vb.VlasovError):
        vb.vlasov_init(1, (8, 8), (1, -1, -1, 1), 0.1)
    vb.vlasov_free()
    with pytest.raises(vb.VlasovError) as e:
        vb.vlasov_step(1)
    assert e.value.code == vb.ENOTINIT
    vb.vlasov_init(1, (8, 8), (-1, 1, -1, 1), 0.1)
    with pytest.raises(vb.VlasovError) as e:
        vb.vlasov_step(0)
    assert e.value.code == vb.EINVAL
    vb.vlasov_free()


@pytest.mark.parametrize("grid", [(353, 61), (64, 48), (1000, 137)])
@pytest.mark.parametrize("bc_p", [BC_ZERO, BC_PERIODIC])
@pytest.mark.parametrize("tile", [0, 2])
def test_history_single_steps_and_ragged_grids(grid, bc_p, tile):
    """The history off the one-pass path on ragged grids, with either momentum boundary, in calls of one, two and three steps
    (a call of one step is a single pass with one half shift: its stored state IS the end-of-step state)."""
    dom = (-PI, PI, -4.0, 4.0)
    f0 = smooth_state(grid[0], grid[1], dom, seed=9)
    o, g = pair(MODEL_HMF, grid, dom, 0.1, f0, bc_p=bc_p, gpu_params=dict(history=1, tune_tile=tile))
    for n in (1, 2, 3, 1):
        g.step(n)
        h = g.history(n)
        for k in range(n):
            o.step(1)
            mo = o.moments()
            assert np.max(np.abs(h[k] - mo)) <= TOL * max(1.0, np.max(np.abs(mo))), (n, k)
    assert rel_err(g.download(), o.download()) <= TOL
    g.close()


@pytest.mark.parametrize("tile", [0, 2])
def test_history_fp32_state_on_the_one_pass_path(tile):
    """fp32 storage: the history off the one-pass path (row sums from the tile kernel, tile = 0, or by the read pass behind the
    warp-specialised kernel, tile = 2; Fourier factors from the fp64 weights)."""
    c = inputs.config("cfg1", n=192)
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=8)
    o.upload(c["f0"])
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], precision=32, history=1, tune_tile=tile)
    g.upload(c["f0"].astype(np.float32))
    g.step(12)
    h = g.history(12)
    for k in range(12):
        o.step(1)
        assert np.max(np.abs(h[k] - o.moments())) <= 1e-4, k
    g.close()


@pytest.mark.parametrize("tile", [1, 2])
def test_fp32_path_matches_oracle_to_1e_4(tile):
    """tile = 1: the tile kernel of small grids, tile = 2: the warp-specialised kernel of the large ones (fp32: both in
    difference form)."""
    c = inputs.config("cfg5", ntheta=600, npts=280)
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=8)
    o.upload(c["f0"])
    o.step(100)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], precision=32, tune_tile=tile)
    g.upload(c["f0"])
    assert g.info()["onepass_tile"] == (1 if tile == 1 else 0)
    g.step(100)
    assert rel_err(g.download().astype(np.float64), o.download()) <= 1e-4
    g.close()


# ----------------------------------------------------------------------------- fourth-order splitting (NEXT #4)
@pytest.mark.parametrize("name,kw,steps", [("cfg1", dict(), 100), ("cfg2", dict(ntheta=256, npts=320), 40),
                                           ("cfg3", dict(ntheta=320, npts=256), 40), ("cfg4", dict(ntheta=512, npts=300), 40),
                                           ("cfg5", dict(ntheta=1500, npts=700), 20)])
def test_order4_steps_match_oracle(name, kw, steps):
    """ORDER = 4 (triple jump of the paper's step, middle sub-step backwards in time): state and
    moments against the oracle's composition, same tolerances as the second-order path"""
    c = inputs.config(name, **kw)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], order=4, **c["params"])
    o.step(steps)
    g.step(steps)
    fo, fg = o.download(), g.download()
    assert rel_err(fg, fo) <= TOL
    mo, mg = o.moments(), g.moments()
    assert np.max(np.abs(mg - mo)) <= TOL * max(1.0, np.max(np.abs(mo)))
    assert mg[0] == pytest.approx(steps * c["dt"])
    g.close()


def test_order4_differs_from_order2_and_records_history():
    c = inputs.config("cfg1", n=128)
    o, g = pair(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], order=4, gpu_params=dict(history=1))
    g.step(6)
    h = g.history(6)
    f4 = g.download()
    g.close()
    for k in range(6):
        o.step(1)
        assert np.max(np.abs(h[k] - o.moments())) <= TOL, k
    g2 = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"])
    g2.upload(c["f0"])
    g2.step(6)
    assert rel_err(g2.download(), f4) > 1e-6   # really another scheme
    g2.close()


def test_order4_fp32_and_refusals():
    c = inputs.config("cfg5", ntheta=600, npts=280)
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=8, order=4)
    o.upload(c["f0"])
    o.step(30)
    g = vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], precision=32, order=4)
    g.upload(c["f0"])
    g.step(30)
    assert rel_err(g.download().astype(np.float64), o.download()) <= 1e-4
    g.close()
    with pytest.raises(vb.VlasovError):
        vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], order=3)
    with pytest.raises(vb.VlasovError):   # the global-spline variant has no fourth-order path
        vb.Vlasov(c["model"], c["grid"], c["domain"], c["dt"], order=4, spline=vb.SPLINE_GS).step(1)
    vb.vlasov_free()
