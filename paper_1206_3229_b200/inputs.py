"""Seeded synthetic inputs: the five BASELINE.json configurations.

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests,
bench).  It holds none of the method's arithmetic -- no spline, stencil,
force or sweep -- only grid nodes, closed-form initial conditions (PAPER.md
eq (17) L147 water-bag; BASELINE.json perturbed Gaussian) and the noise
generator.  It imports neither ``oracle`` nor the CUDA binding.

Conventions (D3, D7, D8):
  * nodes  x_i = x_min + i*(x_max-x_min)/N, i = 0..N-1 (half-open domain);
  * arrays are float64 [Np, Ntheta], theta fastest;
  * water-bag edges strict (|x| < x0 and |p| < p0); not renormalised;
  * noise: f += amp * max(f) * u, u in [0,1) from a counter-based splitmix64
    keyed by seed + linear index, at every grid point.
"""
from __future__ import annotations

import math

import numpy as np

MODEL_FREE, MODEL_HMF, MODEL_RING, MODEL_SHEET = 0, 1, 2, 3
SEED = 12063229


def nodes(lo: float, hi: float, n: int) -> np.ndarray:
    return lo + np.arange(n, dtype=np.float64) * ((hi - lo) / n)


def splitmix64_uniform(seed: int, count: int) -> np.ndarray:
    """u[k] in [0,1): 53 high bits of splitmix64(seed + k)."""
    with np.errstate(over="ignore"):
        z = (np.arange(count, dtype=np.uint64) + np.uint64(seed)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def waterbag(theta: np.ndarray, p: np.ndarray, theta0: float, p0: float,
             noise: float = 0.0, seed: int = SEED) -> np.ndarray:
    """eq (17): f = 1/(4 theta0 p0) on |theta| < theta0, |p| < p0 (+ seeded noise)."""
    level = 1.0 / (4.0 * theta0 * p0)
    f = np.where((np.abs(p)[:, None] < p0) & (np.abs(theta)[None, :] < theta0), level, 0.0)
    if noise > 0.0:
        u = splitmix64_uniform(seed, f.size).reshape(f.shape)
        f = f + (noise * level) * u
    return np.ascontiguousarray(f, dtype=np.float64)


def perturbed_gaussian(theta: np.ndarray, p: np.ndarray, T: float, alpha: float, mode: int = 1) -> np.ndarray:
    g = np.exp(-p * p / (2.0 * T)) / (2.0 * math.pi * math.sqrt(2.0 * math.pi * T))
    return np.ascontiguousarray((1.0 + alpha * np.cos(mode * theta))[None, :] * g[:, None], dtype=np.float64)


# name -> (model, N (square grid), domain, dt, steps, initial condition spec, params)
_CONFIGS = {
    "cfg1": dict(model=MODEL_HMF, n=256, domain=(-math.pi, math.pi, -4.0, 4.0), dt=0.1, steps=100,
                 ic=("waterbag", 1.0, 1.0, 1e-6)),
    "cfg2": dict(model=MODEL_HMF, n=1024, domain=(-math.pi, math.pi, -5.0, 5.0), dt=0.05, steps=2000,
                 ic=("gaussian", 0.4, 1e-4)),
    "cfg3": dict(model=MODEL_RING, n=2048, domain=(-math.pi, math.pi, -3.0, 3.0), dt=0.05, steps=1000,
                 ic=("waterbag", 1.5, 0.5, 1e-6), eps=0.01),
    "cfg4": dict(model=MODEL_SHEET, n=4096, domain=(-10.0, 10.0, -4.0, 4.0), dt=0.02, steps=2000,
                 ic=("waterbag", 1.0, 0.5, 0.0)),
    "cfg5": dict(model=MODEL_HMF, n=8192, domain=(-math.pi, math.pi, -4.0, 4.0), dt=0.1, steps=200,
                 ic=("waterbag", 1.0, 1.0, 1e-6)),
}


def config(name: str, n: int | None = None, ntheta: int | None = None, npts: int | None = None,
           with_f0: bool = True) -> dict:
    """One of BASELINE.json's configs ("cfg1".."cfg5"), optionally on another grid.

    Returns dict(model, grid=(Ntheta, Np), domain, dt, steps, params, f0).
    cfg5 is the throughput sweep; its N defaults to 8192 (also 2048, 4096, 16384).
    """
    c = dict(_CONFIGS[name])
    nt = ntheta or n or c["n"]
    npp = npts or n or c["n"]
    dom = c["domain"]
    out = dict(name=name, model=c["model"], grid=(nt, npp), domain=dom, dt=c["dt"], steps=c["steps"],
               params={k: c[k] for k in ("eps",) if k in c})
    if with_f0:
        th = nodes(dom[0], dom[1], nt)
        p = nodes(dom[2], dom[3], npp)
        ic = c["ic"]
        if ic[0] == "waterbag":
            out["f0"] = waterbag(th, p, ic[1], ic[2], noise=ic[3])
        else:
            out["f0"] = perturbed_gaussian(th, p, ic[1], ic[2])
    return out


def md_waterbag(n: int, theta0: float, p0: float, seed: int = SEED):
    """N particles drawn uniformly from the water-bag |theta| < theta0, |p| < p0 (eq (17); the
    initial state of the Fig. 4 comparison, L192-L206): theta_i = theta0 (2 u_i - 1), p_i = p0 (2 u'_i - 1) with
    u, u' from the counter-based splitmix64 stream (keys seed + i and seed + N + i).  No method arithmetic."""
    u = splitmix64_uniform(seed, 2 * n)
    theta = theta0 * (2.0 * u[:n] - 1.0)
    p = p0 * (2.0 * u[n:] - 1.0)
    return np.ascontiguousarray(theta), np.ascontiguousarray(p)
