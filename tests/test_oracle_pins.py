"""Pins of the CPU oracle (oracle/) against what the paper and the mathematics fix.

Every test here runs without a GPU.  Nothing in this file touches the CUDA path.
Citations are PAPER.md line + section/equation; P-numbers refer to DESIGN.md section 4.
"""
from __future__ import annotations

import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import optimize, special

import oracle
from oracle import BC_PERIODIC, BC_ZERO, MODEL_FREE, MODEL_HMF, MODEL_RING, MODEL_SHEET, Oracle
from paper_1206_3229_b200 import inputs

PI = math.pi


# --------------------------------------------------------------------------- helpers
def read_eq16(golden_dir):
    c = {}
    with open(os.path.join(golden_dir, "eq16_coefficients.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            m, v = line.split()
            c[int(m)] = Fraction(v)
    return c


def fir_weights_exact(c, a: Fraction):
    """Substituting eq (16) into eq (13): f(x) = sum_{m=-4}^{5} w_m f_{k+m}."""
    A = (1 - a) ** 3 - (1 - a)
    B = a ** 3 - a
    w = {}
    for m in range(-4, 6):
        w[m] = (1 - a if m == 0 else 0) + (a if m == 1 else 0) + (A * c.get(m, 0) + B * c.get(m - 1, 0)) / 6
    return w


def run(model, grid, domain, dt, f0, steps=0, threads=4, **params):
    o = Oracle(model, grid, domain, dt, threads=threads, **params)
    o.upload(f0)
    if steps:
        o.step(steps)
    return o


# --------------------------------------------------------------------------- P1: eq (16)
def test_p1_eq16_coefficients_as_printed(golden_dir):
    """Response of the oracle's f'' to a unit impulse = the printed coefficients (L110)."""
    c = read_eq16(golden_dir)
    n = 32
    u = np.zeros(n)
    u[10] = 1.0
    d2 = oracle.fd8_second_derivative(u, 1.0)
    for m in range(-4, 5):
        assert d2[10 - m] == pytest.approx(float(c[m]), rel=1e-15)
    assert np.all(d2[np.abs(np.arange(n) - 10) > 4] == 0.0)
    # 1/h^2 (reading D2): halving h quadruples f''
    assert np.allclose(oracle.fd8_second_derivative(u, 0.5), 4.0 * d2, rtol=1e-15)


def test_p1_fd_exact_on_polynomials_up_to_degree_9():
    n = 17
    x = np.arange(n, dtype=np.float64) - 8.0  # integer nodes: every product below is exact in fp64
    for q in range(0, 10):
        d2 = oracle.fd8_second_derivative(x ** q, 1.0, BC_ZERO)[5:-5]
        exact = q * (q - 1) * x ** max(q - 2, 0) if q >= 2 else np.zeros(n)
        sl = slice(4, n - 4)  # interior: stencil does not reach the zero extension
        scale = max(1.0, np.max(np.abs(x[sl] ** q)))
        assert np.max(np.abs(d2[sl] - exact[sl])) <= 2e-13 * scale, q
    # first failure: degree 10, stencil(x^10)(0) - exact(=0) = -1152 for h = 1  (error -h^8 f^(10)/3150)
    d2 = oracle.fd8_second_derivative(x ** 10, 1.0, BC_ZERO)[5:-5]
    assert d2[8] == pytest.approx(-1152.0, abs=1e-6)
    assert -1152.0 == pytest.approx(-math.factorial(10) / 3150.0)


def test_p1_fd_second_order_scaling_with_h():
    """f'' of sin(kx) on a periodic grid: error = h^8 k^10 / 3150 to leading order."""
    for n in (32, 64):
        h = 2 * PI / n
        x = np.arange(n) * h
        d2 = oracle.fd8_second_derivative(np.sin(x), h)
        err = np.max(np.abs(d2 + np.sin(x)))
        assert err == pytest.approx(h ** 8 / 3150.0, rel=0.05)


# --------------------------------------------------------------------------- P2: a = 0
@pytest.mark.parametrize("bc", [BC_PERIODIC, BC_ZERO])
@pytest.mark.parametrize("cells", [0, 1, -1, 7, -13, 40, -64, 100])
def test_p2_integer_cell_shift_is_bit_exact(bc, cells):
    rng = np.random.default_rng(5)
    n = 64
    u = rng.standard_normal(n)
    h = 0.25  # power of two: -disp/h is an exact integer
    out = oracle.shift_line(u, h, cells * h, bc)  # out_i = u(x_i - cells h) = u_{i - cells}
    idx = np.arange(n) - cells
    if bc == BC_PERIODIC:
        ref = u[idx % n]
    else:
        ref = np.where((idx >= 0) & (idx < n), u[np.clip(idx, 0, n - 1)], 0.0)
    assert np.array_equal(out, ref)


# --------------------------------------------------------------------------- P3: FIR form
@pytest.mark.parametrize("a", [Fraction(1, 2), Fraction(1, 4), Fraction(7, 8), Fraction(1, 1024)])
def test_p3_impulse_response_equals_rational_fir_weights(golden_dir, a):
    c = read_eq16(golden_dir)
    w = fir_weights_exact(c, a)
    n, k0 = 40, 20
    u = np.zeros(n)
    u[k0] = 1.0
    out = oracle.shift_line(u, 1.0, -float(a), BC_PERIODIC)  # u = +a: s = 0, fraction a
    for m in range(-4, 6):
        assert out[k0 - m] == pytest.approx(float(w[m]), rel=1e-13, abs=1e-18), m
    mask = np.ones(n, bool)
    mask[k0 - 5:k0 + 5] = False
    assert np.all(out[mask] == 0.0)


def test_p3_printed_values_of_the_weights(golden_dir):
    """Hand-checkable rationals (P3) and the symmetry w_m(a) = w_{1-m}(1-a)."""
    c = read_eq16(golden_dir)
    w = fir_weights_exact(c, Fraction(1, 2))
    assert w[0] == w[1] == Fraction(3329, 5760)
    assert w[-1] == w[2] == Fraction(-7, 80)
    assert w[-2] == w[3] == Fraction(11, 1008)
    assert w[-3] == w[4] == Fraction(-17, 11520)
    assert w[-4] == w[5] == Fraction(1, 8960)
    a = Fraction(1, 4)
    wa, wb = fir_weights_exact(c, a), fir_weights_exact(c, 1 - a)
    for m in range(-4, 6):
        assert wa[m] == wb[1 - m]
    assert wa[-4] == Fraction(1, 10240) and wa[5] == Fraction(1, 14336)


# --------------------------------------------------------------------------- P4: cubics
@pytest.mark.parametrize("a", [0.5, 0.25, 0.9, 0.013])
def test_p4_one_shift_is_exact_on_cubics(a):
    n = 64
    x = np.arange(n, dtype=np.float64)
    poly = lambda t: 0.3 * t ** 3 - 2.0 * t ** 2 + 5.0 * t - 7.0
    out = oracle.shift_line(poly(x), 1.0, -(3 + a), BC_ZERO)  # out_i = poly(x_i + 3 + a) in the interior
    sl = slice(8, n - 12)
    ref = poly(x + 3 + a)
    assert np.max(np.abs(out[sl] - ref[sl])) <= 1e-12 * np.max(np.abs(ref[sl]))


def test_p4_quartic_defect_at_half_cell():
    """sum m^4 w_m - a^4 = -5/16 at a = 1/2 (P4): the spline is NOT exact on quartics."""
    n = 64
    x = np.arange(n, dtype=np.float64) - 32.0
    out = oracle.shift_line(x ** 4, 1.0, -0.5, BC_ZERO)
    assert out[32] - 0.5 ** 4 == pytest.approx(-5.0 / 16.0, abs=1e-10)


# --------------------------------------------------------------------------- P5: Fourier symbol
def fourier_symbol(kappa, a):
    chat = -205 / 72 + 2 * (8 / 5 * np.cos(kappa) - 1 / 5 * np.cos(2 * kappa) + 8 / 315 * np.cos(3 * kappa)
                            - 1 / 560 * np.cos(4 * kappa))
    A = (1 - a) ** 3 - (1 - a)
    B = a ** 3 - a
    return (1 - a) + a * np.exp(1j * kappa) + (A + B * np.exp(1j * kappa)) * chat / 6


@pytest.mark.parametrize("n,mode", [(64, 1), (64, 5), (256, 1), (256, 16)])
def test_p5_fourier_mode_is_multiplied_by_the_symbol(n, mode):
    kappa = 2 * PI * mode / n
    i = np.arange(n)
    for cells in (0.37, -2.81, 11.5):
        s = math.floor(cells)
        a = cells - s
        S = fourier_symbol(kappa, a)
        re = oracle.shift_line(np.cos(kappa * i), 1.0, -cells)
        im = oracle.shift_line(np.sin(kappa * i), 1.0, -cells)
        ref = S * np.exp(1j * kappa * (i + s))
        assert np.max(np.abs(re + 1j * im - ref)) < 5e-14
        assert abs(S) <= 1 + 1e-15  # stability
    # accuracy of the scheme itself against the exact shift (P5 numbers)
    a = np.linspace(0, 1, 201)
    dev = np.max(np.abs(fourier_symbol(2 * PI / 256, a) - np.exp(1j * 2 * PI / 256 * a)))
    assert dev == pytest.approx(4.7e-9, rel=0.05)


# --------------------------------------------------------------------------- P6/P7: conservation
def test_p6_periodic_line_sum_is_conserved_to_roundoff():
    rng = np.random.default_rng(11)
    u = rng.random(200)
    for cells in (0.123, -7.77, 1234.5):
        out = oracle.shift_line(u, 0.1, cells * 0.1)
        assert abs(out.sum() - u.sum()) < 1e-12 * u.sum()


def test_p6_p7_zero_extension_mass_and_first_moment():
    """Compact data away from the edges: sum conserved; mean index moves by exactly the displacement."""
    n = 200
    i = np.arange(n, dtype=np.float64)
    u = np.exp(-0.5 * ((i - 100) / 6.0) ** 2)
    for cells in (3.3, -12.75):
        out = oracle.shift_line(u, 1.0, cells, BC_ZERO)
        assert abs(out.sum() - u.sum()) < 1e-13 * u.sum()
        assert (i * out).sum() / out.sum() - (i * u).sum() / u.sum() == pytest.approx(cells, abs=1e-11)


@pytest.mark.parametrize("model,domain", [(MODEL_HMF, (-PI, PI, -4, 4)), (MODEL_RING, (-PI, PI, -4, 4)),
                                          (MODEL_SHEET, (-8, 8, -4, 4))])
def test_p7_total_momentum_and_mass_are_conserved(model, domain):
    n = 64
    th = inputs.nodes(domain[0], domain[1], n)
    p = inputs.nodes(domain[2], domain[3], n)
    f0 = np.exp(-0.5 * (p[:, None] - 0.3) ** 2 / 0.09) * np.exp(-0.5 * (th[None, :] - 0.4) ** 2 / 0.5)
    f0 /= f0.sum() * (th[1] - th[0]) * (p[1] - p[0])
    o = run(model, (n, n), domain, 0.05, f0)
    m0 = o.moments()
    # sum_i rho_i F_i = 0 for all three discrete forces (HMF, sheet: identically; ring: K[N-m] = -K[m]
    # holds to the rounding of sin/cos of the table, |K| <= 19.2)
    assert abs(np.dot(o.density(), o.force())) < 2e-13
    o.step(10)
    m1 = o.moments()
    assert m1[1] == pytest.approx(m0[1], rel=1e-11)   # mass
    assert m1[2] == pytest.approx(m0[2], abs=2e-11)   # P
    assert m1[0] == pytest.approx(0.5)


def test_p7_p_sweep_moves_column_momentum_by_F_dt():
    n = 48
    dom = (-PI, PI, -4.0, 4.0)
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = np.exp(-0.5 * p[:, None] ** 2 / 0.2) * (1 + 0.5 * np.cos(th[None, :]))
    o = run(MODEL_FREE, (n, n), dom, 0.1, f0)
    F = 0.8 * np.sin(2 * th) + 0.1
    o.p_sweep(0.1, force=F)
    f1 = o.download()
    pbar0 = (p[:, None] * f0).sum(0) / f0.sum(0)
    pbar1 = (p[:, None] * f1).sum(0) / f1.sum(0)
    assert np.max(np.abs(pbar1 - pbar0 - F * 0.1)) < 1e-11


# --------------------------------------------------------------------------- P8: free streaming
def test_p8_free_streaming_matches_analytic_solution_within_symbol_bound():
    n, mode, b, dt, steps = 128, 2, 0.3, 0.1, 25
    dom = (-PI, PI, -4.0, 4.0)
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    g = np.exp(-0.5 * p ** 2) / math.sqrt(2 * PI)
    f0 = (1 + b * np.cos(mode * th))[None, :] * g[:, None]
    o = run(MODEL_FREE, (n, n), dom, dt, f0, steps=steps)
    t = dt * steps
    exact = (1 + b * np.cos(mode * (th[None, :] - p[:, None] * t))) * g[:, None]
    err = np.max(np.abs(o.download() - exact))
    a = np.linspace(0, 1, 401)
    kappa = 2 * PI * mode / n
    per_shift = np.max(np.abs(fourier_symbol(kappa, a) - np.exp(1j * kappa * a)))
    bound = 2 * steps * b * g.max() * per_shift
    assert err <= bound * 1.0001 + 1e-14
    assert err > 1e-3 * bound  # the bound is not vacuous: the error really is of this origin
    assert o.moments()[0] == pytest.approx(t)


def test_p8_sign_of_the_theta_shift():
    """Positive p moves structure towards larger theta (f(theta - p t)); catches a flipped sign."""
    n = 64
    dom = (-PI, PI, 0.0, 2.0)
    th = inputs.nodes(dom[0], dom[1], n)
    f0 = np.tile(np.exp(-0.5 * (th / 0.3) ** 2), (n, 1))
    o = run(MODEL_FREE, (n, n), dom, 0.5, f0, steps=1)
    f1 = o.download()
    p = inputs.nodes(dom[2], dom[3], n)
    peak = th[np.argmax(f1, axis=1)]
    assert np.max(np.abs(peak - p * 0.5)) <= (th[1] - th[0]) * 0.5 + 1e-12


def test_p8_sign_of_the_p_shift():
    """Positive force moves structure towards larger p (f(p - F dt))."""
    n = 64
    dom = (-PI, PI, -4.0, 4.0)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = np.tile(np.exp(-0.5 * (p / 0.4) ** 2)[:, None], (1, n))
    o = run(MODEL_FREE, (n, n), dom, 0.5, f0)
    F = np.linspace(-2, 2, n)
    o.p_sweep(0.5, force=F)
    f1 = o.download()
    peak = p[np.argmax(f1, axis=0)]
    assert np.max(np.abs(peak - F * 0.5)) <= (p[1] - p[0]) * 0.5 + 1e-12


# --------------------------------------------------------------------------- P9/P10: HMF Gaussian
def test_p9_homogeneous_gaussian_is_stationary():
    n = 64
    dom = (-PI, PI, -5.0, 5.0)
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = inputs.perturbed_gaussian(th, p, 0.4, 0.0)
    o = run(MODEL_HMF, (n, n), dom, 0.05, f0)
    assert np.max(np.abs(o.force())) < 1e-16
    o.step(20)
    assert np.max(np.abs(o.download() - f0)) < 1e-14 * f0.max() * 20
    m = o.moments()
    assert abs(m[5]) < 1e-15 and abs(m[6]) < 1e-15
    assert m[1] == pytest.approx(1.0, abs=1e-9)           # mass of the normalised Gaussian
    assert m[3] == pytest.approx(0.2, abs=1e-8)           # K = T/2
    assert m[4] == pytest.approx(0.5, abs=1e-8)           # U = (1 - M^2)/2


def test_p10_cfg2_initial_moments():
    c = inputs.config("cfg2", n=128)
    o = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"])
    m = o.moments()
    assert m[5] == pytest.approx(5.0e-5, rel=1e-9)        # Mx = alpha/2
    assert abs(m[6]) < 1e-16                              # My = 0 (discrete orthogonality)
    rho = o.density()
    th = inputs.nodes(-PI, PI, 128)
    assert np.allclose(rho, (1 + 1e-4 * np.cos(th)) / (2 * PI), rtol=1e-9)
    assert np.allclose(o.force(), -5.0e-5 * np.sin(th), atol=1e-15)


# --------------------------------------------------------------------------- P11: linear theory
def hmf_growth_rate(T):
    """Root of 2T = 1 - sqrt(pi) z exp(z^2) erfc(z), lambda = z sqrt(2T) (DESIGN.md A.3)."""
    g = lambda z: 1 - math.sqrt(PI) * z * special.erfcx(z) - 2 * T
    return optimize.brentq(g, 1e-12, 50.0) * math.sqrt(2 * T)


def fit_growth(T, n=256, dt=0.1, t0=20.0, t1=50.0):
    dom = (-PI, PI, -5.0, 5.0)
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    o = run(MODEL_HMF, (n, n), dom, dt, inputs.perturbed_gaussian(th, p, T, 1e-4), threads=8)
    ts, ms = [], []
    for k in range(int(round(t1 / dt))):
        o.step(1)
        m = o.moments()
        ts.append(m[0])
        ms.append(math.hypot(m[5], m[6]))
    ts, ms = np.array(ts), np.array(ms)
    sel = ts >= t0
    return np.polyfit(ts[sel], np.log(ms[sel]), 1)[0], ms


def test_p11_dispersion_relation_values_and_threshold():
    assert hmf_growth_rate(0.4) == pytest.approx(0.116166, abs=2e-6)
    assert hmf_growth_rate(0.1) == pytest.approx(0.525573, abs=2e-6)
    assert hmf_growth_rate(0.49) == pytest.approx(0.011315, abs=2e-6)
    with pytest.raises(ValueError):  # no unstable root above T = 1/2
        hmf_growth_rate(0.5001)


def test_p11_growth_rate_at_T_0p4_matches_linear_theory():
    lam, ms = fit_growth(0.4)
    assert lam == pytest.approx(hmf_growth_rate(0.4), rel=0.02)
    assert ms[-1] > 20 * ms[0]


def test_p11_stable_above_threshold_T_0p6():
    lam, ms = fit_growth(0.6, t1=40.0)
    assert ms.max() <= ms[0] * 1.05  # Landau damped: |M| never grows above its initial value
    assert lam < 0.0


# --------------------------------------------------------------------------- P12: the paper's HMF water-bag
def test_p12_paper_waterbag_energy_and_magnetisation(golden_dir):
    vals = {}
    with open(os.path.join(golden_dir, "hmf_waterbag_L192.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            vals[k] = float(v)
    n = 512
    dom = (0.0, 2 * PI, -vals["p_max"], vals["p_max"])
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = np.where((th[None, :] >= vals["theta_lo"]) & (th[None, :] <= vals["theta_hi"])
                  & (np.abs(p)[:, None] <= vals["p0"]), 1.0, 0.0)
    f0 /= f0.sum() * (th[1] - th[0]) * (p[1] - p[0])  # unit mass, as the paper's <.> averages assume
    m = run(MODEL_HMF, (n, n), dom, 0.1, f0).moments()
    assert m[1] == pytest.approx(1.0, rel=1e-12)
    assert math.hypot(m[5], m[6]) == pytest.approx(vals["M"], abs=3e-3)   # printed M = 0.8
    assert m[7] == pytest.approx(vals["e"], abs=5e-3)                     # printed e = 0.7
    # a wrong convention (U = 1 - M^2, or K = p^2) would give 0.88 or 1.22: far outside the tolerance


# --------------------------------------------------------------------------- P13: sheet
def test_p13_sheet_force_of_a_uniform_slab_exact_rationals():
    n, lo, hi = 40, 11, 22  # slab of 12 nodes
    dx = 0.5
    mass = Fraction(3, 4)
    cnt = hi - lo + 1
    rho = np.zeros(n)
    rho[lo:hi + 1] = float(mass / cnt / Fraction(1, 2))
    F = oracle.force_from_rho(MODEL_SHEET, rho, -10.0, -10.0 + n * dx)
    for i in range(n):
        if i < lo:
            ref = mass
        elif i > hi:
            ref = -mass
        else:
            ref = mass * (1 - Fraction(2 * (i - lo) + 1, cnt))
        assert F[i] == pytest.approx(float(ref), abs=1e-15), i


def test_p13_sheet_waterbag_energy_0p375_and_force_profile():
    n = 512
    c = inputs.config("cfg4", n=n)
    o = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"])
    m = o.moments()
    e0 = m[7] / m[1] ** 2 * 1.0  # U scales with mass^2, K with mass; mass = 1 + O(Delta)
    assert m[1] == pytest.approx(1.0, abs=0.03)
    assert m[3] / m[1] == pytest.approx(0.5 ** 2 / 6, rel=0.05)          # K = p0^2/6, O(Delta p / p0)
    assert m[4] / m[1] ** 2 == pytest.approx(1.0 / 3.0, rel=0.03)        # U = x0/3
    assert e0 == pytest.approx(0.375, abs=0.02)
    x = inputs.nodes(-10, 10, n)
    F = o.force() / m[1]
    inside = np.abs(x) < 0.9
    assert np.max(np.abs(F[inside] + x[inside])) < 0.03                  # F = -x/x0 inside
    assert np.allclose(F[x > 1.1], -1.0, atol=1e-12) and np.allclose(F[x < -1.1], 1.0, atol=1e-12)


# --------------------------------------------------------------------------- P14: ring
def test_p14_ring_force_equals_brute_force_trig_double_loop():
    n, eps = 24, 0.05
    rng = np.random.default_rng(3)
    rho = rng.random(n)
    dth = 2 * PI / n
    th = -PI + np.arange(n) * dth
    ref = np.zeros(n)
    for i in range(n):
        for k in range(n):
            if k != i:
                d = th[i] - th[k]
                ref[i] += -math.sin(d) / (2 * math.sqrt(2) * (1 - math.cos(d) + eps) ** 1.5) * rho[k] * dth
    F = oracle.force_from_rho(MODEL_RING, rho, -PI, PI, eps)
    assert np.max(np.abs(F - ref)) < 1e-13 * np.max(np.abs(ref))


def test_p14_ring_force_tends_to_hmf_force_for_large_softening():
    n, eps = 64, 1.0e6
    th = inputs.nodes(-PI, PI, n)
    rho = (1 + 0.4 * np.cos(th - 0.7) + 0.2 * np.sin(3 * th)) / (2 * PI)
    Fr = oracle.force_from_rho(MODEL_RING, rho, -PI, PI, eps) * 2 * math.sqrt(2) * (1 + eps) ** 1.5
    Fh = oracle.force_from_rho(MODEL_HMF, rho, -PI, PI)
    assert np.max(np.abs(Fr - Fh)) < 1e-5 * np.max(np.abs(Fh))


def test_p14_ring_waterbag_closed_form():
    """Uniform slab |theta| < theta0: F(theta) = [V(theta - theta0) - V(theta + theta0)] / (2 theta0)."""
    n, eps, th0 = 4096, 0.01, 1.5
    th = inputs.nodes(-PI, PI, n)
    rho = np.where(np.abs(th) < th0, 1.0 / (2 * th0), 0.0)
    F = oracle.force_from_rho(MODEL_RING, rho, -PI, PI, eps)
    V = lambda x: -1.0 / (math.sqrt(2) * np.sqrt(1 - np.cos(x) + eps))
    ref = (V(th - th0) - V(th + th0)) / (2 * th0)
    sel = np.abs(np.abs(th) - th0) > 0.05
    assert np.max(np.abs(F[sel] - ref[sel])) < 2e-2
    i14 = int(round((1.4 + PI) / (2 * PI / n)))
    assert F[i14] == pytest.approx(-1.75730, abs=2e-2)


def test_p14_ring_potential_table_from_point_masses():
    """V(0) = -1/(sqrt2 sqrt(eps)) = -7.07107 and V(pi) = -1/(sqrt2 sqrt(2 + eps)) = -0.498755 (eq (2), eps =
    0.01) read back from the ORACLE's potential energy: with all the density in one column k, rho_i = c delta_ik,
    U = (1/2) dtheta^2 c^2 V(0); with two equal columns half a circle apart U = dtheta^2 c^2 (V(0) + V(pi))."""
    n, npp, eps = 64, 16, 0.01
    dom = (-PI, PI, -1.0, 1.0)
    dth, dp = 2 * PI / n, 2.0 / npp
    f = np.zeros((npp, n))
    f[:, 5] = 1.0
    c = npp * dp                      # rho_5 = dp * sum_j f = 2
    U1 = run(MODEL_RING, (n, npp), dom, 0.1, f, eps=eps).moments()[4]
    V0 = 2.0 * U1 / (dth * c) ** 2
    assert V0 == pytest.approx(-7.07107, abs=1e-5)
    f[:, 5 + n // 2] = 1.0
    U2 = run(MODEL_RING, (n, npp), dom, 0.1, f, eps=eps).moments()[4]
    Vpi = U2 / (dth * c) ** 2 - V0
    assert Vpi == pytest.approx(-0.498755, abs=1e-6)


def test_p14_ring_potential_energy_of_waterbag():
    n = 512
    c = inputs.config("cfg3", n=n)
    c["f0"][:] = np.where(c["f0"] > 0.1, c["f0"].max(), 0.0)
    m = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], eps=0.01).moments()
    assert m[4] / m[1] ** 2 == pytest.approx(-0.953259, rel=0.01)
    assert m[3] / m[1] == pytest.approx(0.5 ** 2 / 6, rel=0.02)


# --------------------------------------------------------------------------- P15: Strang is second order
def test_p15_strang_splitting_is_second_order():
    n = 64
    dom = (-PI, PI, -5.0, 5.0)
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = inputs.perturbed_gaussian(th, p, 0.4, 0.3)

    def M_at_1(dt):
        o = run(MODEL_HMF, (n, n), dom, dt, f0, steps=int(round(1.0 / dt)))
        return o.moments()[5]

    ref = M_at_1(1.0 / 64)
    e1, e2, e3 = (abs(M_at_1(dt) - ref) for dt in (0.5, 0.25, 0.125))
    assert 3.3 < e1 / e2 < 4.8 and 3.3 < e2 / e3 < 4.8


# --------------------------------------------------------------------------- P21: fourth-order composition (NEXT #4)
def test_p21_triple_jump_composition_is_fourth_order():
    """order = 4 (refs [31], [44]; D23): on smooth data the error of M_x(t = 1) against a fine-step
    run falls by 2^4 per halving of dt (a wrong coefficient, a missing sub-step or a Lie-split ordering gives 4 or 2),
    and it is far below the second-order step's at the same dt."""
    n = 256  # fine enough for the interpolation error (1e-7 here) to stay below the time-splitting error
    dom = (-PI, PI, -5.0, 5.0)
    th = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = inputs.perturbed_gaussian(th, p, 0.4, 0.3)

    def M_at_1(dt, order):
        o = run(MODEL_HMF, (n, n), dom, dt, f0, steps=int(round(1.0 / dt)), threads=8, order=order)
        return o.moments()[5]

    ref = M_at_1(1.0 / 128, 4)
    e1, e2, e3 = (abs(M_at_1(dt, 4) - ref) for dt in (1.0, 0.5, 0.25))
    assert 10.0 < e1 / e2 < 24.0 and 10.0 < e2 / e3 < 24.0, (e1, e2, e3)
    assert e3 < 0.1 * abs(M_at_1(0.25, 2) - ref)


def test_p21_order4_step_is_three_strang_steps_with_the_triple_jump_coefficients():
    """S4(dt) = S2(g1 dt) S2(g2 dt) S2(g1 dt) with g1 = 1/(2 - 2^(1/3)), g2 = 1 - 2 g1 (so that 2 g1 + g2 = 1 and
    2 g1^3 + g2^3 = 0): composed here from three second-order oracles whose dt is set from the closed form."""
    g1 = 1.0 / (2.0 - 2.0 ** (1.0 / 3.0))
    g2 = 1.0 - 2.0 * g1
    assert abs(2 * g1 ** 3 + g2 ** 3) < 1e-15 and g2 < 0
    c = inputs.config("cfg1", ntheta=48, npts=40)
    o4 = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], steps=2, order=4)
    f4, t4 = o4.download(), o4.moments()[0]  # the oracle is a singleton: read it before the next one is made
    f = c["f0"]
    for _ in range(2):
        for g in (g1, g2, g1):
            f = run(c["model"], c["grid"], c["domain"], g * c["dt"], f, steps=1).download()
    assert np.max(np.abs(f4 - f)) <= 1e-15 * np.max(np.abs(f))
    assert t4 == pytest.approx(2 * c["dt"])


def test_p21_order4_free_streaming_moves_by_p_dt():
    """F = 0: the three sub-steps displace row j by (2 g1 + g2) p_j dt = p_j dt in all; against the analytic
    f0(theta - p t, p) on one Fourier mode (a sub-step with a wrong sign or weight misses by O(1))"""
    n, npp = 128, 16
    dom = (-PI, PI, -2.0, 2.0)
    th, p = inputs.nodes(dom[0], dom[1], n), inputs.nodes(dom[2], dom[3], npp)
    f0 = 1.0 + 0.5 * np.cos(th)[None, :] * np.ones(npp)[:, None]
    out = run(MODEL_FREE, (n, npp), dom, 0.7, f0, steps=3, order=4).download()
    ref = 1.0 + 0.5 * np.cos(th[None, :] - p[:, None] * 2.1)
    assert np.max(np.abs(out - ref)) < 1e-6


# --------------------------------------------------------------------------- P16: zero extension
@pytest.mark.parametrize("cells", [0.4, -3.6, 9.25, -70.5, 200.0])
def test_p16_zero_extension_equals_periodic_on_padded_line(cells):
    rng = np.random.default_rng(17)
    n, pad = 60, 300
    u = rng.standard_normal(n)
    out = oracle.shift_line(u, 0.3, cells * 0.3, BC_ZERO)
    big = np.zeros(n + 2 * pad)
    big[pad:pad + n] = u
    ref = oracle.shift_line(big, 0.3, cells * 0.3, BC_PERIODIC)[pad:pad + n]
    assert np.max(np.abs(out - ref)) <= 1e-15 * np.max(np.abs(u))
    if abs(cells) >= n + 5:
        assert np.all(out == 0.0)


def test_p16_fd_zero_extension_is_nonzero_just_outside():
    u = np.ones(12)
    d2 = oracle.fd8_second_derivative(u, 1.0, BC_ZERO)  # indices -5 .. 16
    assert d2[0] == 0.0 and d2[1] == pytest.approx(-1 / 560) and d2[-1] == 0.0
    assert d2[5] == pytest.approx(-205 / 72 + 8 / 5 - 1 / 5 + 8 / 315 - 1 / 560)


# --------------------------------------------------------------------------- P17: drift on cfg 1
@pytest.mark.parametrize("noise", [False, True])
def test_p17_cfg1_drift_bounds(noise):
    c = inputs.config("cfg1")
    if not noise:  # the seeded noise sits on every node, also at the open p edges, where it leaks out
        c["f0"] = np.where(c["f0"] > 0.1, 0.25, 0.0)
    o = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], threads=8)
    m0 = o.moments()
    assert m0[5] / m0[1] == pytest.approx(math.sin(1.0), abs=0.02)        # M0 = sin(1)/1 up to O(Delta)
    worst = 0.0
    for _ in range(100):
        o.step(1)
        m = o.moments()
        worst = max(worst, abs(m[7] - m0[7]) / abs(m0[7]))
    assert m[1] == pytest.approx(m0[1], rel=1e-6 if noise else 1e-12)
    assert m[2] == pytest.approx(m0[2], abs=1e-6 if noise else 1e-12)
    assert worst < 1e-3  # paper Table 2 (L158-L165): 3e-4 .. 5e-4 at dt = 0.1


# --------------------------------------------------------------------------- composition of the step
def test_step_is_theta_half_force_p_full_theta_half():
    """oracle_step == the four stages of section 3 (L71-L87) called one by one, with the force taken
    AFTER the first half advection (eq (10) uses f^(I))."""
    c = inputs.config("cfg1", n=48)
    a2 = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"], steps=3)
    fa = a2.download()
    b = run(c["model"], c["grid"], c["domain"], c["dt"], c["f0"])
    for _ in range(3):
        b.theta_sweep(0.5 * c["dt"])
        F = b.force()
        b.p_sweep(c["dt"], force=F)
        b.theta_sweep(0.5 * c["dt"])
    assert np.array_equal(fa, b.download())


def test_density_and_moments_of_a_known_state():
    n_t, n_p = 32, 40
    dom = (-PI, PI, -2.0, 2.0)
    th = inputs.nodes(dom[0], dom[1], n_t)
    p = inputs.nodes(dom[2], dom[3], n_p)
    f0 = np.ones((n_p, n_t)) * (1 + 0.5 * np.cos(th))[None, :] * (1 + 0.25 * p)[:, None]
    o = run(MODEL_HMF, (n_t, n_p), dom, 0.1, f0)
    dp = 4.0 / n_p
    sp = np.sum(1 + 0.25 * p) * dp
    assert np.allclose(o.density(), (1 + 0.5 * np.cos(th)) * sp, rtol=1e-14)
    m = o.moments()
    assert m[1] == pytest.approx(2 * PI * sp, rel=1e-14)
    assert m[2] == pytest.approx(2 * PI * np.sum(p * (1 + 0.25 * p)) * dp, rel=1e-13)
    assert m[3] == pytest.approx(2 * PI * np.sum(0.5 * p * p * (1 + 0.25 * p)) * dp, rel=1e-13)
    assert m[5] == pytest.approx(0.5 * PI * sp, rel=1e-13) and abs(m[6]) < 1e-14
    assert m[4] == pytest.approx(0.5 * (m[1] ** 2 - m[5] ** 2), rel=1e-13)
    assert m[7] == m[3] + m[4]


# ----------------------------------------------------------------------------- Casimirs (eq (18))
def test_p19_casimirs_of_a_gaussian_closed_form():
    """f = exp(-p^2/2T) / (2 pi sqrt(2 pi T)) (mass 1):  S = -int f log f = log(2 pi sqrt(2 pi T)) + 1/2,
    int f^2 = 1 / (4 pi sqrt(pi T)); the rectangle rule is spectrally accurate for it."""
    T = 0.4
    c = inputs.config("cfg2", n=256)
    th = inputs.nodes(c["domain"][0], c["domain"][1], 256)
    p = inputs.nodes(c["domain"][2], c["domain"][3], 256)
    f0 = np.exp(-p[:, None] ** 2 / (2 * T)) / (2 * PI * math.sqrt(2 * PI * T)) * np.ones_like(th)[None, :]
    o = run(MODEL_HMF, (256, 256), c["domain"], 0.05, f0)
    S, C2, neg, fmax = o.casimirs()
    assert S == pytest.approx(math.log(2 * PI * math.sqrt(2 * PI * T)) + 0.5, abs=1e-12)
    assert C2 == pytest.approx(1.0 / (4 * PI * math.sqrt(PI * T)), rel=1e-12)
    assert neg == 0.0
    assert fmax == pytest.approx(1.0 / (2 * PI * math.sqrt(2 * PI * T)), rel=1e-15)


def test_p19_casimirs_of_a_waterbag_and_of_signed_values():
    """Noise-free water-bag of height f0 on n nodes: S = -n f0 log f0 dx dp, int f^2 = n f0^2 dx dp (exact counts);
    a state with negative values: those nodes add nothing to S and their sum is the negative mass (D20)."""
    c = inputs.config("cfg4", n=64)  # sheet water-bag, no noise
    f0 = c["f0"]
    h = float(f0.max())
    n = int(np.count_nonzero(f0))
    assert n > 0 and np.all((f0 == 0) | (f0 == h))
    dxdp = (c["domain"][1] - c["domain"][0]) / 64 * (c["domain"][3] - c["domain"][2]) / 64
    o = run(c["model"], c["grid"], c["domain"], c["dt"], f0)
    S, C2, neg, fmax = o.casimirs()
    assert S == pytest.approx(-n * h * math.log(h) * dxdp, rel=1e-14)
    assert C2 == pytest.approx(n * h * h * dxdp, rel=1e-14)
    assert neg == 0.0 and fmax == h
    g = f0.copy()
    g[3, 5] = -0.25
    g[7, 9] = -0.5
    o = run(c["model"], c["grid"], c["domain"], c["dt"], g)
    S2, C22, neg2, _ = o.casimirs()
    assert S2 == pytest.approx(S, rel=1e-14)                      # f[3,5], f[7,9] were 0 before: no change
    assert neg2 == pytest.approx(-0.75 * dxdp, rel=1e-14)
    assert C22 == pytest.approx(C2 + (0.0625 + 0.25) * dxdp, rel=1e-14)


def test_p19_casimirs_invariant_under_integer_cell_shifts_and_bounded_drift():
    """An integer-cell shift permutes the values along each line: every Casimir is unchanged (to the round-off of
    the sums).  A fractional shift of smooth data changes S and C2 only at the order of the interpolation error;
    int f^2 cannot grow beyond round-off for a periodic constant shift (|symbol| <= 1, pin P5)."""
    n_t, n_p = 96, 64
    dom = (-PI, PI, -3.0, 3.0)
    th = inputs.nodes(dom[0], dom[1], n_t)
    p = inputs.nodes(dom[2], dom[3], n_p)
    f0 = np.exp(-p[:, None] ** 2) * (1.2 + np.cos(th)[None, :])
    dx = 2 * PI / n_t
    o = run(MODEL_FREE, (n_t, n_p), dom, 0.0, f0, bc_p=BC_PERIODIC)
    base = o.casimirs()
    o.p_sweep(1.0, force=np.full(n_t, -5 * 6.0 / n_p))          # five cells along p, periodic
    after = o.casimirs()
    assert np.allclose(after, base, rtol=1e-14, atol=0)
    o2 = run(MODEL_FREE, (n_t, n_p), dom, 0.0, f0)
    o2.theta_sweep(0.37 * dx)                                   # displacement p * 0.37 dx: fractional for most rows
    a2 = o2.casimirs()
    assert a2[1] <= base[1] * (1 + 1e-14)
    assert abs(a2[0] - base[0]) < 1e-6 * abs(base[0]) and abs(a2[1] - base[1]) < 1e-6 * base[1]


# ----------------------------------------------------------------------------- the paper's own sheet runs (Table 2)
def paper_sheet_state(n):
    """Set-up of PAPER.md L145-L150: x, p in [-2, 2], water-bag of eq (17) with x0 = 1, p0 = 0.5, edges included."""
    dom = (-2.0, 2.0, -2.0, 2.0)
    x = inputs.nodes(dom[0], dom[1], n)
    p = inputs.nodes(dom[2], dom[3], n)
    f0 = np.where((np.abs(x)[None, :] <= 1.0) & (np.abs(p)[:, None] <= 0.5), 0.5, 0.0)
    return dom, f0


def test_p20_energy_error_of_the_papers_sheet_run_matches_table_2(golden_dir):
    """Table 2 (L158-L165) prints delta e = 5e-4 for n = 256 at dt = 0.1 with the FD interpolation.  The oracle, run
    with the paper's own boundary conditions (periodic in x and p, L113) to t = 100, shows 4.9e-4: same value to
    the one digit the paper prints (the run length is not stated, D13: asserted within a factor 2).  Its norm is
    conserved to round-off where the paper reports 4e-5 (D14: the telescoping sum is exact)."""
    rows = [ln.split() for ln in open(os.path.join(golden_dir, "sheet_table2_L158.txt")) if not ln.startswith("#")]
    table = {int(r[0]): (float(r[1]), float(r[2])) for r in rows}
    n = 256
    dom, f0 = paper_sheet_state(n)
    o = run(MODEL_SHEET, (n, n), dom, 0.1, f0, threads=os.cpu_count() or 4, bc_x=BC_PERIODIC, bc_p=BC_PERIODIC)
    m0 = o.moments()
    s0 = o.casimirs()[0]
    de = dn = 0.0
    for _ in range(100):
        o.step(10)
        m = o.moments()
        de = max(de, abs(m[7] - m0[7]) / abs(m0[7]))
        dn = max(dn, abs(m[1] - m0[1]) / m0[1])
    assert 0.5 * table[n][0] <= de <= 2.0 * table[n][0]
    assert dn <= 1e-12 <= table[n][1]
    # Fig. 2 (L180): the entropy rises from its initial plateau once filaments reach the mesh size
    assert o.casimirs()[0] > s0 + 0.2


# --------------------------------------------------------------------------- G1-G7: Global Spline, system (15)
# the paper's comparator "GS" (L100-L104, Tables 1-2).  DESIGN.md section 4.
SQRT3 = math.sqrt(3.0)


def test_g1_gs_second_derivative_solves_system_15_and_has_the_closed_form_impulse_response():
    """(a) residual of the system as read in D22 (2/3 on the diagonal) on random data; (b) the response to a unit
    impulse is sqrt(3) r^|k| convolved with (1, -2, 1)/h^2, r = sqrt(3) - 2: the textbook inverse of the
    constant-coefficient operator (1/6, 2/3, 1/6); (c) a constant line has f'' = 0 and the sum of f'' over a
    periodic line is 0 (telescoping right-hand side, unit row sums): the mass of a shifted line is conserved."""
    rng = np.random.default_rng(15)
    n, h = 97, 0.37
    u = rng.standard_normal(n)
    d2 = oracle.vlasov_oracle.gs_second_derivative(u, h)
    res = (np.roll(d2, -1) / 6 + 2 * d2 / 3 + np.roll(d2, 1) / 6) * h * h - (np.roll(u, -1) - 2 * u + np.roll(u, 1))
    assert np.abs(res).max() < 1e-13
    assert abs(d2.sum()) < 1e-11
    assert np.abs(oracle.vlasov_oracle.gs_second_derivative(np.full(n, 3.7), h)).max() == 0.0
    e = np.zeros(n)
    e[40] = 1.0
    g = oracle.vlasov_oracle.gs_second_derivative(e, 1.0)
    r = SQRT3 - 2.0
    k = np.arange(-40, n - 40)
    G = SQRT3 * r ** np.abs(k).astype(float)
    want = np.zeros(n)
    for i in range(n):
        want[i] = (SQRT3 * r ** abs(k[i] + 1.0)) - 2 * G[i] + (SQRT3 * r ** abs(k[i] - 1.0))
    assert np.abs(g - want).max() < 1e-14


@pytest.mark.parametrize("n,mode", [(64, 1), (64, 5), (100, 17), (33, 16)])
def test_g2_gs_second_derivative_fourier_symbol(n, mode):
    """On e^{i kappa k} system (15) gives f'' = -(2 (1 - cos kappa)/h^2) * 3/(2 + cos kappa) f."""
    h = 0.2
    kap = 2 * PI * mode / n
    k = np.arange(n)
    lam = -(2 * (1 - math.cos(kap)) / h ** 2) * 3.0 / (2.0 + math.cos(kap))
    for u in (np.cos(kap * k), np.sin(kap * k)):
        d2 = oracle.vlasov_oracle.gs_second_derivative(u, h)
        assert np.abs(d2 - lam * u).max() < 1e-11 * abs(lam)


@pytest.mark.parametrize("disp", [0.1, -0.23, 1.9, -7.3, 0.37 * 4])
def test_g3_gs_shift_equals_scipy_periodic_cubic_spline(disp):
    """The periodic interpolating cubic spline is unique: a GS shift = scipy's CubicSpline(bc_type='periodic')
    evaluated at the feet x_i - disp (a library routine the oracle does not use)."""
    from scipy.interpolate import CubicSpline

    rng = np.random.default_rng(3)
    n, h = 50, 0.37
    u = rng.standard_normal(n)
    cs = CubicSpline(np.arange(n + 1) * h, np.append(u, u[0]), bc_type="periodic")
    out = oracle.shift_line(u, h, disp, BC_PERIODIC, oracle.SPLINE_GS)
    ref = cs((np.arange(n) * h - disp) % (n * h))
    assert np.abs(out - ref).max() < 1e-13
    if disp == 0.37 * 4:  # integer-cell shift: bit-exact copy (P2 holds for any f'')
        assert np.array_equal(oracle.shift_line(u, 1.0, 4.0, BC_PERIODIC, oracle.SPLINE_GS), np.roll(u, 4))


def test_g4_gs_first_derivative_is_continuous_across_knots_fd_is_not():
    """The defining condition of (15) (L100): one-sided slopes at a knot agree for GS on rough data; with the
    local f'' of eq (16) they do not (the FD spline is only C0 there)."""
    rng = np.random.default_rng(4)
    n, h, e = 40, 1.0, 1e-6
    u = rng.standard_normal(n)

    def jump(spline):
        right = (oracle.shift_line(u, h, -e, BC_PERIODIC, spline) - u) / e   # (f(x_i + e) - f(x_i)) / e
        left = (u - oracle.shift_line(u, h, e, BC_PERIODIC, spline)) / e     # (f(x_i) - f(x_i - e)) / e
        return np.abs(right - left).max()

    assert jump(oracle.SPLINE_GS) < 1e-4      # O(e f'') + round-off / e
    assert jump(oracle.SPLINE_FD) > 1e-2


def test_g5_gs_zero_extension_equals_periodic_on_padded_line_and_conserves_the_line_sum():
    rng = np.random.default_rng(5)
    n, h, pad = 60, 0.5, 120
    u = np.zeros(n)
    u[20:40] = rng.random(20)
    up = np.concatenate([np.zeros(pad), u, np.zeros(pad)])
    for disp in (0.1, -3.3, 5.2):
        a = oracle.shift_line(u, h, disp, BC_ZERO, oracle.SPLINE_GS)
        b = oracle.shift_line(up, h, disp, BC_PERIODIC, oracle.SPLINE_GS)[pad:pad + n]
        assert np.abs(a - b).max() < 1e-15
    out = oracle.shift_line(rng.standard_normal(77), 0.3, 0.123, BC_PERIODIC, oracle.SPLINE_GS)
    # mass: sum of f'' is 0 (G1), alpha + beta = 1
    v = rng.standard_normal(77)
    assert abs(oracle.shift_line(v, 0.3, 0.123, BC_PERIODIC, oracle.SPLINE_GS).sum() - v.sum()) < 1e-12
    assert out.shape == (77,)


def test_g6_gs_shift_symbol_and_cubic_exactness():
    """A GS shift multiplies e^{i kappa k} by (1-a) + a e^{i kappa} + ((A + B e^{i kappa})/6) * lambda h^2 with
    lambda of G2; and on a periodic line the shift of a smooth mode converges at fourth order."""
    n, h, a = 64, 1.0, 0.3
    k = np.arange(n)
    for mode in (1, 3, 9):
        kap = 2 * PI * mode / n
        lam = -(2 * (1 - math.cos(kap))) * 3.0 / (2.0 + math.cos(kap))
        A, B = (1 - a) ** 3 - (1 - a), a ** 3 - a
        S = (1 - a) + a * np.exp(1j * kap) + (A + B * np.exp(1j * kap)) / 6 * lam
        c = oracle.shift_line(np.cos(kap * k), h, -a * h, BC_PERIODIC, oracle.SPLINE_GS)
        s = oracle.shift_line(np.sin(kap * k), h, -a * h, BC_PERIODIC, oracle.SPLINE_GS)
        got = c + 1j * s
        assert np.abs(got - S * np.exp(1j * kap * k)).max() < 1e-13
    errs = []
    for n in (32, 64):
        x = 2 * PI * np.arange(n) / n
        hh = 2 * PI / n
        out = oracle.shift_line(np.sin(x), hh, 0.5 * hh, BC_PERIODIC, oracle.SPLINE_GS)
        errs.append(np.abs(out - np.sin(x - 0.5 * hh)).max())
    assert 14.0 < errs[0] / errs[1] < 18.0


def test_g7_gs_energy_error_of_the_papers_sheet_run_matches_table_2(golden_dir):
    """Table 2 (L158-L165), GS columns, dt = 0.1: delta e = 4e-4 at n = 512 and 2e-4 at n = 256.  The oracle with
    KEY_SPLINE = GS and the paper's periodic boundaries, run to t = 100 (run length unstated, D13), shows 5.2e-4
    and 4.9e-4: within a factor 2 of the print at 512 (asserted), a factor 2.4 at 256 (asserted within 3; the FD
    and GS errors of the oracle agree to 1e-6 there, as they do in the paper's rows 512-2048: at dt = 0.1 the
    error is the splitting error, not the interpolation)."""
    rows = [ln.split() for ln in open(os.path.join(golden_dir, "sheet_table2_gs_L158.txt")) if not ln.startswith("#")]
    table = {int(r[0]): (float(r[1]), float(r[2])) for r in rows}
    for n, fac in ((512, 2.0), (256, 3.0)):
        dom, f0 = paper_sheet_state(n)
        o = run(MODEL_SHEET, (n, n), dom, 0.1, f0, threads=os.cpu_count() or 4, bc_x=BC_PERIODIC, bc_p=BC_PERIODIC,
                spline=oracle.SPLINE_GS)
        m0 = o.moments()
        de = dn = 0.0
        for _ in range(100):
            o.step(10)
            m = o.moments()
            de = max(de, abs(m[7] - m0[7]) / abs(m0[7]))
            dn = max(dn, abs(m[1] - m0[1]) / m0[1])
        assert table[n][0] / fac <= de <= fac * table[n][0]
        assert dn <= 1e-12
