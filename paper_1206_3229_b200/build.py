"""Build step: compile the CUDA library in-tree with nvcc for sm_100a.

    python -m paper_1206_3229_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The resulting ``csrc/libvlasov_b200.so`` is git-ignored but travels
with the working tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(CSRC, "libvlasov_b200.so")
SOURCES = [os.path.join(CSRC, "vlasov_api.cu"), os.path.join(CSRC, "hmf_md.cu"), os.path.join(CSRC, "hmf_noalloc.cu")]
DEPS = SOURCES + [os.path.join(CSRC, h) for h in ("vlasov_kernels.cuh", "vlasov_theta_bulk.cuh", "vlasov_ptx.cuh", "vlasov_fused.cuh", "vlasov_fused_ws.cuh", "vlasov_tile.cuh", "vlasov_gs.cuh")] + [
    os.path.join(ROOT, "include", "vlasov.h"), os.path.join(ROOT, "include", "hmf_md.h"), os.path.join(ROOT, "include", "hmf_noalloc.h")]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build_library(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-shared", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-o", tmp] + SOURCES
    extra = os.environ.get("VLASOV_NVCC_FLAGS")
    if extra:
        cmd[1:1] = extra.split()
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
