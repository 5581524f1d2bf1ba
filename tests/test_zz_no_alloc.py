"""hmf_noalloc_moments (include/hmf_noalloc.h): the entry point that allocates nothing (its scratch memory is a
file-scope `static __device__` array) against the existing path hmf_md_moments (scratch from cudaMalloc), on the same
device arrays, on several calls in a row that share the scratch array.  The two differ in the order in which the
particles are added up (4096 per block and the blocks in index order on the device, against a grid-stride loop and a
host sum): 1e-12 on the moments, the tolerance tests/test_gpu_md.py uses for them.

This file is collected last on purpose (pytest -x stops at the first failure)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_1206_3229_b200 import binding as vb
from paper_1206_3229_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-12


def noalloc_moments(md, t, out_dev):
    import torch

    stream = torch.cuda.current_stream(md.device).cuda_stream
    vb.hmf_noalloc_moments(md.theta_dev.data_ptr(), md.p_dev.data_ptr(), md.n, t, out_dev.data_ptr(), stream)
    torch.cuda.synchronize()
    return out_dev.cpu().numpy()


@pytest.mark.parametrize("n", [1, 4096, 4097, 100003, 1000003])
def test_no_alloc_moments_match_the_allocating_path_on_calls_in_a_row(n):
    import torch

    th, p = inputs.md_waterbag(n, 1.2, 0.7)
    md = vb.HmfMd(n, 0.1)
    try:
        md.upload(th, p)
        out_dev = torch.full((8,), float("nan"), dtype=torch.float64, device=md.device)
        for call in range(3):  # the state moves between the calls; the scratch array keeps what the call before left
            want = md.moments()
            got = noalloc_moments(md, want[0], out_dev)
            assert np.all(np.isfinite(got))
            assert np.max(np.abs(got - want)) <= TOL * max(1.0, np.max(np.abs(want))), (call, got, want)
            md.step(2)
        # two calls back to back on one stream without a host synchronisation in between: the second result stands
        want = md.moments()
        stream = torch.cuda.current_stream(md.device).cuda_stream
        out2 = torch.zeros(8, dtype=torch.float64, device=md.device)
        vb.hmf_noalloc_moments(md.theta_dev.data_ptr(), md.p_dev.data_ptr(), md.n, 1.0, out_dev.data_ptr(), stream)
        vb.hmf_noalloc_moments(md.theta_dev.data_ptr(), md.p_dev.data_ptr(), md.n, want[0], out2.data_ptr(), stream)
        torch.cuda.synchronize()
        a, b = out_dev.cpu().numpy(), out2.cpu().numpy()
        assert a[0] == 1.0 and np.array_equal(a[1:], b[1:])  # same inputs, same scratch: bit-identical
        assert np.max(np.abs(b - want)) <= TOL * max(1.0, np.max(np.abs(want)))
    finally:
        md.close()


def test_no_alloc_after_a_larger_call_a_smaller_one_is_not_polluted():
    """the partial sums of a call with many blocks stay in the scratch array; a call with fewer blocks must not read them"""
    import torch

    big, small = 300000, 5000
    th, p = inputs.md_waterbag(big, 1.0, 1.0)
    md = vb.HmfMd(big, 0.1)
    try:
        md.upload(th, p)
        out_dev = torch.zeros(8, dtype=torch.float64, device=md.device)
        noalloc_moments(md, 0.0, out_dev)
        stream = torch.cuda.current_stream(md.device).cuda_stream
        vb.hmf_noalloc_moments(md.theta_dev.data_ptr(), md.p_dev.data_ptr(), small, 0.0, out_dev.data_ptr(), stream)
        torch.cuda.synchronize()
        got = out_dev.cpu().numpy()
    finally:
        md.close()
    md = vb.HmfMd(small, 0.1)
    try:
        md.upload(th[:small], p[:small])
        want = md.moments()
    finally:
        md.close()
    assert np.max(np.abs(got - want)) <= TOL * max(1.0, np.max(np.abs(want)))


def test_no_alloc_rejects_sizes_beyond_its_scratch_array_and_bad_arguments():
    import torch

    buf = torch.zeros(16, dtype=torch.float64, device="cuda:0")
    out = torch.full((8,), 7.0, dtype=torch.float64, device="cuda:0")
    for n in (vb.NOALLOC_MAX_PARTICLES + 1, 2 * vb.NOALLOC_MAX_PARTICLES, 0, -5):
        with pytest.raises(vb.VlasovError) as ei:
            vb.hmf_noalloc_moments(buf.data_ptr(), buf.data_ptr(), n, 0.0, out.data_ptr(), 0)
        assert ei.value.code == vb.EINVAL
    assert "exceeds the maximum" in str(ei.value) or "n must be" in str(ei.value)
    with pytest.raises(vb.VlasovError):
        vb.hmf_noalloc_moments(0, buf.data_ptr(), 8, 0.0, out.data_ptr(), 0)
    torch.cuda.synchronize()
    assert np.all(out.cpu().numpy() == 7.0)  # nothing was launched


def test_no_alloc_entry_point_really_does_not_allocate():
    """free device memory as the driver reports it does not move across calls (after the first one, which loads the
    module and looks up the symbol), and the source names no allocating call"""
    import os

    import torch

    n = 200000
    th, p = inputs.md_waterbag(n, 1.0, 1.0)
    md = vb.HmfMd(n, 0.1)
    try:
        md.upload(th, p)
        out_dev = torch.zeros(8, dtype=torch.float64, device=md.device)
        noalloc_moments(md, 0.0, out_dev)
        free0, _ = torch.cuda.mem_get_info(md.device)
        for _ in range(20):
            noalloc_moments(md, 0.0, out_dev)
        free1, _ = torch.cuda.mem_get_info(md.device)
        assert free0 - free1 < (1 << 20)  # twenty calls that each allocated their 256 KiB of partial sums would show
    finally:
        md.close()
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = open(os.path.join(root, "paper_1206_3229_b200", "csrc", "hmf_noalloc.cu")).read()
    code = "\n".join(line.split("//")[0] for line in src.splitlines())
    for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "new ", "malloc(", "std::vector"):
        assert word not in code, word
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256)" in code
