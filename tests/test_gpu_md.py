"""Parity of the CUDA molecular dynamics of the HMF model (include/hmf_md.h, md_kick_drift_kernel; SURVEY.md 8(f)
NEXT #3; eqs (7)-(8), L206) against the CPU oracle (oracle/hmf_md_oracle.c), particle by particle, through
the C ABI.  The two differ in rounding only (libm's sin/cos against CUDA's sincos, summation order of M, the fused
half drifts between steps); the N-body dynamics amplifies that by a few orders of magnitude over 100 steps, hence
1e-9 on theta and p (observed 1e-12) and 1e-12 on the moments."""
from __future__ import annotations

import numpy as np
import pytest

from oracle import MdOracle
from paper_1206_3229_b200 import binding as vb
from paper_1206_3229_b200 import inputs

pytestmark = pytest.mark.gpu


def both(n, dt, steps, theta0=1.0, p0=1.0, chunks=None):
    th, p = inputs.md_waterbag(n, theta0, p0)
    o = MdOracle(n, dt)
    o.upload(th, p)
    o.step(steps)
    tho, po = o.download()
    mo = o.moments()
    o.close()
    g = vb.HmfMd(n, dt)
    g.upload(th, p)
    for c in (chunks or [steps]):
        g.step(c)
    thg, pg = g.download()
    mg = g.moments()
    g.close()
    return tho, po, mo, thg, pg, mg


@pytest.mark.parametrize("n", [1, 2, 31, 1000, 1025, 40000, 1000003])
def test_md_100_steps_match_oracle(n):
    steps = 100 if n <= 40000 else 20
    tho, po, mo, thg, pg, mg = both(n, 0.1, steps)
    assert np.max(np.abs(thg - tho)) <= 1e-9 and np.max(np.abs(pg - po)) <= 1e-9
    assert np.max(np.abs(mg - mo)) <= 1e-12 * max(1.0, np.max(np.abs(mo)))
    assert mg[0] == pytest.approx(steps * 0.1)


@pytest.mark.parametrize("scale", [3.0, 2.0e3, 9.0e4, 4.0e6])
def test_md_trigonometry_at_large_angles(scale):
    """theta is never wrapped (reading D24), so the kernel's sine and cosine (the library's sincos for the kick, a small-angle
    rotation of it for the sums of the drifted angles) must hold at whatever angles a run reaches: the sums of cos theta_i
    and sin theta_i of angles spread over [-scale, scale] against numpy (libm), and one step against the oracle.
    (A hand-written sincos -- reduction by pi/2 in three doubles and Taylor polynomials -- passed this test and was NOT
    faster than the library's: 48.2 against 49.5 G particle-steps/s; not kept.)"""
    n = 20011
    rng = np.random.default_rng(7)
    th = rng.uniform(-scale, scale, n)
    th[:8] = [0.0, scale, -scale, 0.5 * np.pi, -0.5 * np.pi, np.pi, 0.25 * np.pi * 3, 1e-300]
    p = rng.uniform(-1.0, 1.0, n)
    g = vb.HmfMd(n, 0.1)
    g.upload(th, p)
    m = g.moments()
    # moments: [t, M_x, M_y, ...]: M = (1/N) sum (cos, sin)
    assert abs(m[1] - np.mean(np.cos(th))) <= 2e-15 and abs(m[2] - np.mean(np.sin(th))) <= 2e-15
    g.step(1)
    thg, pg = g.download()
    g.close()
    o = MdOracle(n, 0.1)
    o.upload(th, p)
    o.step(1)
    tho, po = o.download()
    o.close()
    # theta += c dt p is one FMA on the GPU and a product and a sum in the oracle: the angles may differ by an ulp of theta
    # (9e-10 at 4e6), and through M so do the kicks (observed 2.5e-13 at scale 4e6, 1e-16 at scale 3)
    assert np.max(np.abs(thg - tho)) <= 1e-15 * max(1.0, scale)
    assert np.max(np.abs(pg - po)) <= 1e-14 + 2e-19 * scale


def test_md_steps_per_call_do_not_matter_beyond_rounding():
    """step(7) + step(3) against step(10): the half drifts between steps are fused inside a call and separate across
    calls (theta += c dt p twice against theta += 2 c dt p once)"""
    a = both(5000, 0.1, 10)
    b = both(5000, 0.1, 10, chunks=[7, 3])
    assert np.max(np.abs(a[3] - b[3])) <= 1e-12 and np.max(np.abs(a[4] - b[4])) <= 1e-12


def test_md_is_reproducible_and_counts_its_launches():
    outs = []
    for _ in range(2):
        th, p = inputs.md_waterbag(300000, 1.0, 1.0)
        g = vb.HmfMd(300000, 0.1)
        g.upload(th, p)
        l0 = vb.hmf_md_launch_count()
        g.step(12)
        assert vb.hmf_md_launch_count() - l0 == 3 * 12 + 1
        outs.append(g.download())
        g.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_md_conserves_energy_and_momentum_at_the_papers_time_step():
    """dt = 0.1 (L206): energy error of the fourth-order integrator below 1e-6, momentum to round-off, over 200 steps
    of a million particles; the magnetisation relaxes from its water-bag value sin(1)/1"""
    n = 1 << 20
    th, p = inputs.md_waterbag(n, 1.0, 1.0)
    g = vb.HmfMd(n, 0.1, attach=False)       # library-owned buffers
    g.upload(th, p)
    m0 = g.moments()
    g.step(200)
    m1 = g.moments()
    g.close()
    assert m0[1] == pytest.approx(np.sin(1.0), abs=3e-3)
    assert abs(m1[5] - m0[5]) < 1e-6 and abs(m1[6] - m0[6]) < 1e-14
    assert abs(m1[1] - m0[1]) > 0.01


def test_md_errors():
    with pytest.raises(vb.VlasovError):
        vb.HmfMd(0, 0.1)
    g = vb.HmfMd(10, 0.1)
    with pytest.raises(vb.VlasovError):
        g.step(0)
    g.close()
    with pytest.raises(vb.VlasovError) as e:
        g.step(1)
    assert e.value.code == vb.ENOTINIT
