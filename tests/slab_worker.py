"""Worker of test_slab_sharding.py (torch.distributed.run, gloo, CPU): every rank advances its p-slab with the sharded
stepper of paper_1206_3229_b200/slab.py on the oracle stand-in and writes its owned rows to DIST_OUT."""
from __future__ import annotations

import os
import sys

import numpy as np
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
from paper_1206_3229_b200 import inputs, slab  # noqa: E402
from slab_oracle_backend import OracleSlab  # noqa: E402


def main() -> int:
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    name, nt, npp, steps, halo = os.environ["SLAB_CFG"], int(os.environ["SLAB_NT"]), int(os.environ["SLAB_NP"]), int(
        os.environ["SLAB_STEPS"]), int(os.environ["SLAB_HALO"])
    c = inputs.config(name, ntheta=nt, npts=npp)
    b = OracleSlab(c["model"], c["grid"], c["domain"], c["dt"], rank, world, halo, **c["params"])
    b.upload_global(c["f0"])
    dp = (c["domain"][3] - c["domain"][2]) / npp
    st = slab.SlabStepper(b, rank, world, dist, check_halo=lambda fmax: slab.halo_depth(fmax, c["dt"], dp))
    st.step(steps)
    np.save(os.path.join(os.environ["DIST_OUT"], "slab_rank%d.npy" % rank), b.download_owned())
    b.close()
    dist.barrier()
    dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
