"""p-slab sharding: the host side on CPU ranks (gloo), the library's slab mode on one GPU.

CPU: world_size 2 and 3 under torch.distributed.run: partition, density all-reduce and halo exchange of
paper_1206_3229_b200/slab.py, with the oracle standing in for the library, against the unsharded oracle.
GPU (one device, the context is a singleton): the library's slab mode, rank after rank -- each rank's slab is advanced
through the stage calls with the halos and the density that the OTHER slabs would have sent taken from an unsharded
library run -- against the oracle."""
from __future__ import annotations

import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from oracle import Oracle
from paper_1206_3229_b200 import inputs, slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_and_halo_arithmetic():
    for n, w in ((10, 3), (8192, 8), (7, 7), (100, 1)):
        rows = [slab.slab_rows(n, w, r) for r in range(w)]
        assert rows[0][0] == 0 and rows[-1][1] == n
        assert all(rows[r][1] == rows[r + 1][0] for r in range(w - 1))
        assert max(b - a for a, b in rows) - min(b - a for a, b in rows) <= 1
    assert slab.halo_depth(0.84, 0.1, 8.0 / 8192) == 87 + 6          # cfg 5 at 8192^2: 86.02 cells
    d = slab.slab_domain((-1.0, 1.0, -4.0, 4.0), 8, 2, 6)
    assert d == (-1.0, 1.0, -2.0, 2.0)


def run_ranks(world, cfg, nt, npp, steps, halo, tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ, DIST_OUT=str(tmp_path), SLAB_CFG=cfg, SLAB_NT=str(nt), SLAB_NP=str(npp), SLAB_STEPS=str(steps),
               SLAB_HALO=str(halo))
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                        "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "tests", "slab_worker.py")],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    return np.concatenate([np.load(tmp_path / ("slab_rank%d.npy" % k)) for k in range(world)], axis=0)


@pytest.mark.parametrize("world,cfg,nt,npp,halo", [(2, "cfg1", 64, 96, 12), (3, "cfg3", 48, 120, 30), (2, "cfg4", 96, 64, 10)])
def test_sharded_steps_equal_the_unsharded_oracle_gloo(world, cfg, nt, npp, halo, tmp_path):
    steps = 6
    f = run_ranks(world, cfg, nt, npp, steps, halo, tmp_path)
    c = inputs.config(cfg, ntheta=nt, npts=npp)
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=2, **c["params"])
    o.upload(c["f0"])
    o.step(steps)
    ref = o.download()
    o.close()
    assert f.shape == ref.shape
    # the slabs evaluate p_j = p_min(slab) + j dp: the same momenta up to one rounding, hence 1e-13 and not bit equality
    assert np.max(np.abs(f - ref)) <= 1e-13 * np.max(np.abs(ref))


def test_too_thin_a_halo_is_refused(tmp_path):
    with pytest.raises(AssertionError) as e:
        run_ranks(2, "cfg3", 48, 120, 2, 7, tmp_path)     # the ring force moves by far more than one row
    assert "too thin" in str(e.value)


# ------------------------------------------------------------------------------------------------ GPU: slab mode
@pytest.mark.gpu
@pytest.mark.parametrize("cfg,nt,npp,world,halo", [("cfg1", 300, 200, 2, 16), ("cfg5", 1024, 768, 3, 24), ("cfg4", 512, 300, 2, 12),
                                                   ("cfg3", 320, 256, 2, 60)])
def test_library_slab_mode_rank_by_rank_matches_oracle(cfg, nt, npp, world, halo):
    """Every rank's slab through the library's stage calls (THETA_HALF, RHO, FORCE_FROM_RHO, P_FULL on rows + halos),
    one rank after the other on the one GPU.  What a rank would receive -- the other slabs' density and its halo rows --
    is computed from the oracle's f_I of the same step, so each slab is checked on its own against the oracle."""
    import torch

    from paper_1206_3229_b200 import binding as vb

    c = inputs.config(cfg, ntheta=nt, npts=npp)
    dp = (c["domain"][3] - c["domain"][2]) / npp
    o = Oracle(c["model"], c["grid"], c["domain"], c["dt"], threads=8, **c["params"])
    o.upload(c["f0"])
    state = c["f0"].copy()
    for step in range(3):
        o.upload(state)
        o.theta_sweep(0.5 * c["dt"])
        f1 = o.download()                         # f_I of this step, all rows
        rho = o.density()
        o.p_sweep(c["dt"])
        o.theta_sweep(0.5 * c["dt"])
        ref = o.download()
        new = np.empty_like(state)
        for rank in range(world):
            b = slab.LibrarySlab(c["model"], c["grid"], c["domain"], c["dt"], rank, world, halo, **c["params"])
            b.upload_global(state)
            b.theta_half()
            mine = b.local_rho().cpu().numpy().copy()
            own = dp * f1[b.j0:b.j1].sum(axis=0)
            assert np.max(np.abs(mine - own)) <= 1e-13 * np.max(np.abs(rho))      # density of the owned rows only
            b.rho.copy_(torch.from_numpy(rho))                                    # "all-reduce"
            fmax = b.force_from_rho()
            assert slab.halo_depth(fmax, c["dt"], dp) <= halo
            f = b.get_state()
            assert f.shape == (b.halo_lo + b.rows + b.halo_hi, nt)
            if b.halo_lo:                                                         # "halo exchange"
                f[:b.halo_lo].copy_(torch.from_numpy(f1[b.j0 - b.halo_lo:b.j0]))
            if b.halo_hi:
                f[b.halo_lo + b.rows:].copy_(torch.from_numpy(f1[b.j1:b.j1 + b.halo_hi]))
            b.p_full()
            b.theta_half()
            new[b.j0:b.j1] = b.download_owned()
            with pytest.raises(vb.VlasovError):
                vb.vlasov_step(1)                                                 # a slab is advanced stage by stage
            b.close()
        assert np.max(np.abs(new - ref)) <= 1e-12 * np.max(np.abs(ref)), step
        state = new
    o.close()
