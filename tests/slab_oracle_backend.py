"""CPU stand-in for the library's slab mode, built on the ORACLE (test infrastructure): lets the sharded sequencing,
partition and exchange plan of paper_1206_3229_b200/slab.py run on CPU ranks (gloo), with the same interface as
``slab.LibrarySlab``.  The slab is an oracle over the owned rows plus the halos."""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_1206_3229_b200 import slab


class OracleSlab:
    def __init__(self, model, grid, domain, dt, rank, world, halo, eps=0.01):
        nt, np_total = int(grid[0]), int(grid[1])
        self.model, self.domain, self.dt, self.eps = model, domain, dt, eps
        self.j0, self.j1 = slab.slab_rows(np_total, world, rank)
        self.rows = self.j1 - self.j0
        self.halo_lo = halo if rank > 0 else 0
        self.halo_hi = halo if rank < world - 1 else 0
        self.dp = (domain[3] - domain[2]) / np_total
        ext = slab.slab_domain(domain, np_total, self.j0 - self.halo_lo, self.j1 + self.halo_hi)
        self.o = oracle.Oracle(model, (nt, self.rows + self.halo_lo + self.halo_hi), ext, dt, threads=1, eps=eps)
        self.F = np.zeros(nt)
        self.rho = torch.zeros(nt, dtype=torch.float64)

    def upload_global(self, f0):
        f = np.zeros((self.rows + self.halo_lo + self.halo_hi, f0.shape[1]))
        f[self.halo_lo:self.halo_lo + self.rows] = f0[self.j0:self.j1]
        self.o.upload(f)

    def download_owned(self):
        return self.o.download()[self.halo_lo:self.halo_lo + self.rows]

    def theta_half(self):
        self.o.theta_sweep(0.5 * self.dt)

    def local_rho(self):
        self.rho[:] = torch.from_numpy(self.dp * self.download_owned().sum(axis=0))
        return self.rho

    def force_from_rho(self):
        self.F = oracle.force_from_rho(self.model, self.rho.numpy().copy(), self.domain[0], self.domain[1], self.eps)
        return float(np.max(np.abs(self.F)))

    def get_state(self):
        return torch.from_numpy(self.o.download())

    def put_state(self, f):
        self.o.upload(f.numpy())

    def p_full(self):
        self.o.p_sweep(self.dt, force=self.F)

    def close(self):
        self.o.close()
