"""p-slab sharding of the Strang step over several GPUs: one process per GPU,
``torch.distributed`` (NCCL over NVLink) for the two exchanges a step has.

Decomposition: rank r owns a contiguous slab of rows (momenta) of the global grid.  Per Strang step
    theta(dt/2)              row-local, no traffic                                     eq (9)
    rho                      local column sums of the owned rows, then ONE all-reduce   eq (10)   (Ntheta doubles)
    F                        from the global rho, replicated on every rank              eqs (7)-(8) / (2) / (4)
    halo exchange            H rows of f_I to each neighbour (H > max|F| dt/dp + 5)
    p(dt)                    over the owned rows and both halos                         eq (11)
    theta(dt/2)              row-local                                                  eq (12)
The arithmetic of every stage runs in the CUDA library (slab mode of include/vlasov.h: VLASOV_KEY_HALO_LO / _HI and the
stage calls of vlasov_substep); this module only sequences the stages and issues the two collectives, which is
argument marshalling of the same kind as binding.py.  It is written against a small backend interface so that the
sequencing, the partition and the exchange plan can be exercised on CPU ranks (gloo) in the tests.

Status: built and tested for correctness (world_size 2 on CPU ranks with gloo; slab mode of the library against the
oracle on one GPU, rank by rank).  No multi-GPU box was available to this build: unmeasured on NVLink.
"""
from __future__ import annotations

import math


def slab_rows(np_total: int, world: int, rank: int):
    """rows [j0, j1) of the global grid that rank owns: an even split, the first np_total % world ranks get one more"""
    base, extra = divmod(int(np_total), int(world))
    j0 = rank * base + min(rank, extra)
    return j0, j0 + base + (1 if rank < extra else 0)


def halo_depth(fmax: float, dt: float, dp: float) -> int:
    """halo rows that keep the owned rows of a momentum shift exact: integer shift + the ten-tap stencil (eq (11), (16))"""
    return int(math.ceil(abs(fmax * dt) / dp)) + 6


def slab_domain(domain, np_total: int, j0: int, j1: int):
    """(x_min, x_max, p_min, p_max) of the rows [j0, j1): same dp as the global grid"""
    dp = (domain[3] - domain[2]) / np_total
    return (domain[0], domain[1], domain[2] + j0 * dp, domain[2] + j1 * dp)


class SlabStepper:
    """Sequences the stages of a sharded Strang step.  ``backend`` provides

        theta_half()                  eq (9) / (12) on the owned rows (leaves the column sums behind)
        local_rho() -> tensor         density of the owned rows, [Ntheta] (may alias library memory)
        force_from_rho()              force from the (all-reduced) density vector; returns max|F| if check is wanted
        get_state() -> tensor         current f, [halo_lo + owned + halo_hi, Ntheta] (may alias device memory)
        put_state(tensor)             hand it back (no-op when get_state aliases)
        p_full()                      eq (11) over all rows of the buffer
        halo_lo, halo_hi, rows        halo depths and owned rows of this rank

    ``dist`` is ``torch.distributed`` (initialised by the caller) or None for a single rank."""

    def __init__(self, backend, rank: int, world: int, dist=None, check_halo=None):
        self.b, self.rank, self.world, self.dist = backend, rank, world, dist
        self.check_halo = check_halo  # callable(max|F|) -> required halo depth, or None
        if world > 1 and dist is None:
            raise ValueError("world > 1 needs torch.distributed")
        if rank > 0 and backend.halo_lo < 1 or rank < world - 1 and backend.halo_hi < 1:
            raise ValueError("an inner slab edge needs a halo")
        if backend.rows < max(backend.halo_lo, backend.halo_hi):
            raise ValueError("slab of %d rows is thinner than its halo: use fewer ranks" % backend.rows)

    # ---- the two exchanges ---------------------------------------------------------------------------------
    def all_reduce_rho(self):
        rho = self.b.local_rho()
        if self.world > 1:
            self.dist.all_reduce(rho)      # sum over the slabs: eq (10) over all momenta
        return rho

    def exchange_halos(self):
        """my first / last owned rows -> the upper / lower halo of the neighbour below / above me"""
        b = self.b
        f = b.get_state()
        lo, n, hi = b.halo_lo, b.rows, b.halo_hi
        ops, keep = [], []
        if self.world > 1:
            P2POp, isend, irecv = self.dist.P2POp, self.dist.isend, self.dist.irecv
            if self.rank > 0:                       # neighbour below (smaller momenta)
                send = f[lo:lo + lo].contiguous()   # as many rows as the neighbour's halo (all inner halos are alike)
                keep.append(send)
                ops.append(P2POp(isend, send, self.rank - 1))
                ops.append(P2POp(irecv, f[0:lo], self.rank - 1))
            if self.rank < self.world - 1:          # neighbour above
                send = f[lo + n - hi:lo + n].contiguous()
                keep.append(send)
                ops.append(P2POp(isend, send, self.rank + 1))
                ops.append(P2POp(irecv, f[lo + n:lo + n + hi], self.rank + 1))
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()
        b.put_state(f)

    # ---- one step ---------------------------------------------------------------------------------------------
    def step(self, n: int = 1):
        b = self.b
        for _ in range(n):
            b.theta_half()                      # eq (9)
            self.all_reduce_rho()               # eq (10)
            fmax = b.force_from_rho()           # eqs (7)-(8) / (2) / (4)
            if self.check_halo is not None and fmax is not None:
                need = self.check_halo(fmax)
                have = min(h for h in (b.halo_lo, b.halo_hi) if h > 0) if (b.halo_lo or b.halo_hi) else need
                if need > have:
                    raise RuntimeError("halo of %d rows is too thin for max|F| = %g (needs %d)" % (have, fmax, need))
            self.exchange_halos()
            b.p_full()                          # eq (11)
            b.theta_half()                      # eq (12)


class _DevVec:
    """a library-owned device vector as something torch can alias (``__cuda_array_interface__``)"""

    def __init__(self, ptr: int, n: int):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 2}


class LibrarySlab:
    """Backend of SlabStepper on the CUDA library: one slab per process / GPU (the context is a singleton)."""

    def __init__(self, model, grid, domain, dt, rank: int, world: int, halo: int, device: str = "cuda:0", **params):
        import torch

        from . import binding as vb

        self.vb, self.torch = vb, torch
        nt, np_total = int(grid[0]), int(grid[1])
        self.j0, self.j1 = slab_rows(np_total, world, rank)
        self.rows = self.j1 - self.j0
        self.halo_lo = halo if rank > 0 else 0
        self.halo_hi = halo if rank < world - 1 else 0
        self.ntheta = nt
        self.g = vb.Vlasov(model, (nt, self.rows), slab_domain(domain, np_total, self.j0, self.j1), dt, device=device,
                           fuse=0, halo_lo=self.halo_lo, halo_hi=self.halo_hi, **params)
        self.rho = torch.as_tensor(_DevVec(vb.vlasov_vector_ptr(vb.VEC_RHO), nt), device=self.g.device)
        self.force = torch.as_tensor(_DevVec(vb.vlasov_vector_ptr(vb.VEC_FORCE), nt), device=self.g.device)

    def upload_global(self, f0):
        self.g.upload(f0[self.j0:self.j1])

    def download_owned(self):
        return self.g.download()

    def theta_half(self):
        self.vb.vlasov_substep(self.vb.SUB_THETA_HALF)

    def local_rho(self):
        self.vb.vlasov_substep(self.vb.SUB_RHO)
        return self.rho

    def force_from_rho(self):
        self.vb.vlasov_substep(self.vb.SUB_FORCE_FROM_RHO)
        return float(self.force.abs().max().item())

    def get_state(self):
        return self.g.current_state_tensor()

    def put_state(self, f):
        pass

    def p_full(self):
        self.vb.vlasov_substep(self.vb.SUB_P_FULL)

    def close(self):
        self.g.close()
