"""Pins of the HMF molecular-dynamics oracle (oracle/hmf_md_oracle.c; PAPER.md L56-L65 eqs
(7)-(8), L206 / Fig. 4, ref. [44]) against what the mathematics fixes independently of it.  All run without a GPU."""
from __future__ import annotations

import math

import numpy as np
import pytest
from scipy.special import ellipk

from oracle import MdOracle, MODEL_HMF, Oracle
from paper_1206_3229_b200 import inputs

PI = math.pi


def md(theta, p, dt, steps=0):
    o = MdOracle(len(theta), dt)
    o.upload(theta, p)
    if steps:
        o.step(steps)
    return o


def test_m1_two_particles_are_a_pendulum_with_the_elliptic_period():
    """N = 2: phi = theta_1 - theta_2 obeys phi'' = -sin(phi) (eq (1) with eq (3): U = (1 - cos phi)/2), whose period
    for the amplitude phi0 is 4 K(sin^2(phi0/2)).  After one period the pair is back (error of the fourth-order
    integrator), after half a period phi = -phi0; the centre of mass moves uniformly."""
    phi0 = 2.0
    T = 4.0 * ellipk(math.sin(phi0 / 2.0) ** 2)
    errs = []
    for nst in (40, 80, 160):
        o = md(np.array([0.3 + phi0 / 2, 0.3 - phi0 / 2]), np.array([0.25, 0.25]), T / nst, nst // 4)
        th, p = o.download()
        errs.append(abs(th[0] - th[1]))          # phi(T/4) = 0, passed at full speed: the error is the phase error
        o.step(nst // 4)
        th, p = o.download()
        assert th[0] - th[1] == pytest.approx(-phi0, abs=1e-6)
        o.step(nst // 2)
        th, p = o.download()
        assert th[0] - th[1] == pytest.approx(phi0, abs=1e-6)
        assert 0.5 * (th[0] + th[1]) == pytest.approx(0.3 + 0.25 * T, abs=1e-12)   # centre of mass: free motion
        assert p[0] + p[1] == pytest.approx(0.5, abs=1e-14)
    assert errs[2] < 1e-5
    assert 12.0 < errs[0] / errs[1] < 20.0 and 12.0 < errs[1] / errs[2] < 20.0    # fourth order


def test_m2_energy_error_is_fourth_order_and_momentum_exact():
    th, p = inputs.md_waterbag(2000, 1.0, 1.0)
    e0 = md(th, p, 0.1).moments()
    de = []
    for dt in (0.4, 0.2, 0.1):
        m = md(th, p, dt, int(round(4.0 / dt))).moments()
        de.append(abs(m[5] - e0[5]))
        assert m[6] == pytest.approx(e0[6], abs=1e-15)   # sum_i F_i = 0 identically: total momentum to round-off
        assert m[0] == pytest.approx(4.0)
    assert 10.0 < de[0] / de[1] < 24.0 and 10.0 < de[1] / de[2] < 24.0
    assert de[2] < 1e-6


def test_m3_potential_energy_is_the_double_sum_of_eq_1():
    th, p = inputs.md_waterbag(300, 2.0, 0.5)
    o = md(th, p, 0.1, 7)
    m = o.moments()
    assert m[4] == pytest.approx(o.potential_double_sum(), abs=1e-14)
    th2, _ = o.download()
    assert m[1] == pytest.approx(np.mean(np.cos(th2)), abs=1e-15) and m[2] == pytest.approx(np.mean(np.sin(th2)), abs=1e-15)
    assert m[3] == pytest.approx(0.5 * np.mean(o.download()[1] ** 2), abs=1e-15)


def test_m4_integrator_is_time_reversible():
    """drift-kick-drift compositions with symmetric coefficients are reversible: forwards, flip p, forwards again
    returns to the start up to rounding (amplified by the chaotic dynamics: 1e-10 after 50 steps)"""
    th, p = inputs.md_waterbag(500, 1.0, 1.0)
    o = md(th, p, 0.1, 50)
    th1, p1 = o.download()
    assert np.max(np.abs(th1 - th)) > 0.1
    o = md(th1, -p1, 0.1, 50)
    th2, p2 = o.download()
    assert np.max(np.abs(th2 - th)) < 1e-10 and np.max(np.abs(p2 + p)) < 1e-10


def test_m5_one_step_is_the_seven_stage_sequence():
    """one step written out here with numpy from the closed-form coefficients (g1 = 1/(2 - 2^(1/3)), g2 = 1 - 2 g1):
    drift g1/2, kick g1, drift (g1+g2)/2, kick g2, drift (g1+g2)/2, kick g1, drift g1/2, force by eq (7)"""
    th, p = inputs.md_waterbag(64, 1.5, 0.7)
    dt = 0.1
    g1 = 1.0 / (2.0 - 2.0 ** (1.0 / 3.0))
    g2 = 1.0 - 2.0 * g1
    a, b = th.copy(), p.copy()
    for c, d in ((g1 / 2, g1), ((g1 + g2) / 2, g2), ((g1 + g2) / 2, g1), (g1 / 2, None)):
        a = a + c * dt * b
        if d is not None:
            mx, my = np.mean(np.cos(a)), np.mean(np.sin(a))
            b = b + d * dt * (-np.sin(a) * mx + np.cos(a) * my)
    tho, po = md(th, p, dt, 1).download()
    assert np.max(np.abs(tho - a)) < 1e-15 and np.max(np.abs(po - b)) < 1e-15


def test_m6_magnetisation_follows_the_vlasov_oracle_within_particle_noise():
    """PAPER.md L206 / Fig. 4: the MD run and the Vlasov solution agree (there: up to t = 70 with N = 2e7).  Here the
    water-bag theta0 = 1, p0 = 1 with N = 2e5 against the Vlasov oracle on a 256 x 256 grid up to t = 4: the two
    M_x(t) differ by less than a few 1/sqrt(N) plus the grid's O(dx) representation of the bag edge."""
    n = 200000
    th, p = inputs.md_waterbag(n, 1.0, 1.0)
    o = md(th, p, 0.1)
    c = inputs.config("cfg1", n=256)
    f0 = c["f0"] / (np.sum(c["f0"]) * (2 * PI / 256) * (8.0 / 256))   # unit mass, as the particles have
    mds = []
    for _ in range(8):
        o.step(5)
        mds.append(o.moments()[1])
    o.close()
    v = Oracle(MODEL_HMF, c["grid"], c["domain"], 0.1, threads=4)
    v.upload(f0)
    for k in range(8):
        v.step(5)
        assert abs(v.moments()[5] - mds[k]) < 0.01, (k, v.moments()[5], mds[k])
    assert max(mds) - min(mds) > 0.05   # M_x really evolves over the window (the bound above is not vacuous)
    v.close()
