"""gene_nl_compute_static: the entry point for callers that cannot allocate device memory.

Some users of this library cannot let it call cudaMalloc: their own pool already owns the whole device, or a
cudaMalloc (which synchronises the device) would stall the other streams of their time step.  For them the library
keeps the intermediate arrays of the planes in flight in a static device array and offers one plan-free call for
planes of 96 x 48 modes (include/gene_nl.h).  This file checks that the call gives what the plan-based path gives,
that it keeps doing so when the shared static array still holds the previous call's data, and that it refuses every
size the array was not laid out for.

The file sorts last on purpose (pytest -x stops at the first failure: a failure here hides no other test), and it
passes both alone in a fresh process (its first call does the per-device set-up) and after the rest of the suite.
"""
import os
import re

import numpy as np
import pytest
import torch

from helpers import TOL, plane_errors, plane_max_errors

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _planes(t, wl):
    from paper_1310_1485_b200 import workloads as W
    return W.as_planes(t, wl).cpu().numpy()


@pytest.mark.gpu
def test_static_entry_point_matches_the_plan_path_on_two_calls_in_a_row(cuda_device):
    from paper_1310_1485_b200 import GeneNL, gene_nl_compute_static, workloads as W

    torch.cuda.set_device(cuda_device)
    # first call: 168 planes over at most 64 slots, so every slot is reused by a second and a third plane;
    # second call: different data and only 30 planes, so 34 slots still hold the first call's Z and P
    cases = (W.small_workload(96, 48, 4, 7, 3, 2, 0.04, 0.04, True, seed=21),
             W.small_workload(96, 48, 5, 3, 2, 1, 0.03, 0.05, True, seed=22, scale=-1.3))
    outs, wants = [], []
    for wl in cases:   # the two static calls back to back on one stream, nothing of the plan path in between
        chi, g, rhs = W.make_inputs(wl, cuda_device)
        out = rhs.clone()
        gene_nl_compute_static(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, chi, g, out, wl.scale)
        outs.append((wl, chi, g, rhs, out))
    torch.cuda.synchronize()
    for wl, chi, g, rhs, out in outs:
        want = rhs.clone()
        with GeneNL(wl) as nl:   # the existing path: plan, cudaMalloc'ed scratch
            nl.compute(chi, g, want)
            torch.cuda.synchronize()
        wants.append(want)
    for (wl, chi, g, rhs, out), want in zip(outs, wants):
        got, ref, r_in = _planes(out, wl), _planes(want, wl), _planes(rhs, wl)
        assert np.isfinite(got).all()
        assert plane_errors(wl, got, ref, r_in).max() <= TOL
        assert plane_max_errors(wl, got, ref, r_in).max() <= TOL
        h = wl.nx0 // 2   # the Nyquist row of rhs is not touched
        assert np.array_equal(got[:, :, h], r_in[:, :, h])
    # accumulating a second time into the same rhs: rhs_in + 2 * scale * N
    wl, chi, g, rhs, out = outs[1]
    gene_nl_compute_static(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, chi, g, out, wl.scale)
    torch.cuda.synchronize()
    got, ref, r_in = _planes(out, wl), _planes(wants[1], wl), _planes(rhs, wl)
    assert plane_errors(wl, got, 2.0 * ref - r_in, r_in).max() <= TOL
    # and the driver sees no allocation: free device memory is the same before and after further calls (the per-device
    # set-up happened in the first call above; no torch allocation between the two readings)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        gene_nl_compute_static(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, chi, g, out, 0.0)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0


def test_static_entry_point_rejects_what_its_scratch_was_not_laid_out_for():
    """Sizes are checked before any CUDA call, so this runs without a GPU."""
    from paper_1310_1485_b200 import GeneNLError, gene_nl_compute_static
    with pytest.raises(GeneNLError, match="96 x 48"):       # a larger plane does not fit a slot
        gene_nl_compute_static(256, 64, 1, 1, 1, 1, 0.1, 0.1, 16, 32, 48, 1.0, stream=0)
    with pytest.raises(GeneNLError, match="96 x 48"):       # a smaller one has no kernel without a plan
        gene_nl_compute_static(16, 8, 1, 1, 1, 1, 0.1, 0.1, 16, 32, 48, 1.0, stream=0)
    with pytest.raises(GeneNLError, match="MAX_PLANES"):    # 2^31 planes
        gene_nl_compute_static(96, 48, 1 << 16, 1 << 15, 1, 1, 0.1, 0.1, 16, 32, 48, 1.0, stream=0)
    with pytest.raises(GeneNLError, match="positive"):
        gene_nl_compute_static(96, 48, 0, 1, 1, 1, 0.1, 0.1, 16, 32, 48, 1.0, stream=0)


def test_static_entry_point_source_allocates_nothing():
    """The translation unit behind the call contains no allocating CUDA call and takes the array's address properly."""
    src = open(os.path.join(ROOT, "paper_1310_1485_b200", "csrc", "gene_nl_static.cu")).read()
    code = re.sub(r"//[^\n]*", "", re.sub(r"/\*.*?\*/", "", src, flags=re.S))
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaStreamCreate", "cudaEventCreate", "std::vector", "malloc(", "new "):
        assert banned not in code, banned
    assert "static __device__ __align__(256)" in code
    assert "cudaGetSymbolAddress" in code
