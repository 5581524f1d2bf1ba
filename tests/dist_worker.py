"""Worker of test_multi_process.py: run under torch.distributed.run with the gloo backend (CPU).

Exercises the host-side N > 1 logic of bench.py: every rank times its own replica, the job time is the MAX over
ranks, and the whole-job value is all replicas' grid points over that time (replicas only,
no data-path collective)."""
from __future__ import annotations

import json
import os
import sys

import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def main() -> int:
    rank, local_rank, world = bench.dist_env()
    dist.init_process_group("gloo")
    assert dist.get_rank() == rank and dist.get_world_size() == world
    local_ms = 10.0 + 5.0 * rank                      # rank r "measured" 10 + 5 r ms
    ms = bench.max_over_ranks(local_ms, world)        # CPU tensor: gloo
    pts, steps = 1000.0, 4
    value = world * pts * steps / (ms * 1e-3) / 1e9
    dist.barrier()
    out = {"rank": rank, "world": world, "ms": ms, "value": value}
    with open(os.path.join(os.environ["DIST_OUT"], "rank%d.json" % rank), "w") as fh:
        json.dump(out, fh)
    dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
