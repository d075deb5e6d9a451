"""Parity of the x-global CUDA kernel (gene_nlx_*, through the C ABI) against the CPU oracle, element by element on
the same seeded inputs; tolerance as for the flux-tube path: per plane ||out - ref||_2 / ||scale pref N||_2 <= 1e-11."""
import numpy as np
import pytest
import torch

import oracle
from helpers import TOL
from paper_1310_1485_b200 import workloads as W

pytestmark = pytest.mark.gpu


def run_gpu(wl, arrs):
    from paper_1310_1485_b200 import gene_nlx_compute, gene_nlx_create, gene_nlx_destroy
    vex, vey, dxg, dyg, pref, rhs = arrs
    out = rhs.clone()
    h = gene_nlx_create(wl.nx, wl.nky0, wl.planes)
    try:
        gene_nlx_compute(h, vex, vey, dxg, dyg, pref, out, wl.scale)
        torch.cuda.synchronize()
    finally:
        gene_nlx_destroy(h)
    return out


def plane_errors(wl, arrs, out, planes):
    vex, vey, dxg, dyg, pref, rhs = arrs
    idx = torch.as_tensor(planes, device=out.device)
    a, b, c, d, r = (t[idx].cpu().numpy() for t in (vex, vey, dxg, dyg, rhs))
    ref = oracle.nlx_pseudospectral(a, b, c, d, pref.cpu().numpy(), r, wl.scale)
    got = out[idx].cpu().numpy()
    num = np.linalg.norm((got - ref).reshape(len(planes), -1), axis=1)
    den = np.linalg.norm((ref - r).reshape(len(planes), -1), axis=1)
    assert np.all(den > 0)
    return num / den


# every instantiated y length, x extents with a ragged tail (not a multiple of the 32-point tile), one plane
@pytest.mark.parametrize("nx,nky0,planes", [(64, 16, 37), (32, 8, 5), (96, 32, 9), (40, 16, 7), (7, 8, 3), (1, 16, 1),
                                            (33, 32, 2), (24, 48, 3), (20, 64, 2), (16, 96, 2), (9, 128, 2)])
def test_small_shapes_all_planes(cuda_device, nx, nky0, planes):
    wl = W.XGlobalWorkload(f"xg_{nx}x{nky0}", nx, nky0, planes, 100 + nx + nky0, 0.7)
    arrs = W.make_xglobal_inputs(wl, cuda_device)
    out = run_gpu(wl, arrs)
    assert plane_errors(wl, arrs, out, np.arange(planes)).max() <= TOL


def test_against_the_definition_and_properties(cuda_device):
    wl = W.XGlobalWorkload("xg_def", 64, 16, 6, 5, 1.0)
    vex, vey, dxg, dyg, pref, rhs = W.make_xglobal_inputs(wl, cuda_device)
    zero = torch.zeros_like(rhs)
    ones = torch.ones_like(pref)
    n = run_gpu(wl, (vex, vey, dxg, dyg, ones, zero)).cpu().numpy()
    for p in range(wl.planes):   # the truncated ky convolution, plane by plane
        ref = oracle.nlx_convolution_plane(*(t[p].cpu().numpy() for t in (vex, vey, dxg, dyg)))
        assert np.linalg.norm(n[p] - ref) <= TOL * np.linalg.norm(ref)
    wl0 = W.XGlobalWorkload("xg_s0", 64, 16, 6, 5, 0.0)
    assert torch.equal(run_gpu(wl0, (vex, vey, dxg, dyg, pref, rhs)), rhs)        # scale = 0: bit-identical
    n2 = run_gpu(wl, (dxg, dyg, vex, vey, ones, zero))                            # the product commutes
    assert np.abs(n2.cpu().numpy() - n).max() <= 1e-13 * np.abs(n).max()
    vex2 = vex.clone()
    vex2[:, 0, :] += 3.0j                                                         # Im of ky = 0 is ignored
    assert torch.equal(run_gpu(wl, (vex2, vey, dxg, dyg, ones, zero)), run_gpu(wl, (vex, vey, dxg, dyg, ones, zero)))


def test_paper_shape_sampled_planes(cuda_device):
    """The paper's plane shape (64 x 16) on enough planes to fill the device several times over."""
    wl = W.XGlobalWorkload("xg_paper_shape", 64, 16, 65536, 9, 0.7)
    arrs = W.make_xglobal_inputs(wl, cuda_device)
    out = run_gpu(wl, arrs)
    rng = np.random.default_rng(0)
    planes = np.unique(np.concatenate([[0, 1, wl.planes - 1], rng.integers(0, wl.planes, 40)]))
    assert plane_errors(wl, arrs, out, planes).max() <= TOL


def test_host_entry_point_streams_chunks_to_the_same_bits(cuda_device):
    """gene_nlx_compute_host (chunks of xy-planes on asynchronous streams): same kernel per chunk, so the
    same bits as the device-resident call; 37 planes = 4 ragged chunks, and enough planes for several 64 MiB chunks."""
    from paper_1310_1485_b200 import gene_nlx_compute_host, gene_nlx_create, gene_nlx_destroy
    for planes in (37, 20000):
        wl = W.XGlobalWorkload("xg_host", 64, 16, planes, 12, 0.7)
        arrs = W.make_xglobal_inputs(wl, cuda_device)
        dev = run_gpu(wl, arrs)
        vex, vey, dxg, dyg, pref, rhs = (t.cpu().pin_memory() for t in arrs)
        h = gene_nlx_create(wl.nx, wl.nky0, wl.planes)
        try:
            gene_nlx_compute_host(h, vex, vey, dxg, dyg, pref, rhs, wl.scale)
            gene_nlx_compute_host(h, vex, vey, dxg, dyg, pref, rhs, 0.0)      # staging buffers are reused; scale 0
        finally:
            gene_nlx_destroy(h)
        assert torch.equal(rhs.to(cuda_device), dev)
    assert plane_errors(wl, arrs, dev, np.array([0, 1, 9999, planes - 1])).max() <= TOL


def test_errors_are_reported(cuda_device):
    from paper_1310_1485_b200 import GeneNLError, gene_nlx_compute, gene_nlx_create, gene_nlx_destroy
    with pytest.raises(GeneNLError):
        gene_nlx_create(64, 7, 1)       # Ny = 21: no kernel
    with pytest.raises(GeneNLError):
        gene_nlx_create(0, 16, 1)
    wl = W.XGlobalWorkload("xg_err", 32, 16, 2, 1, 1.0)
    vex, vey, dxg, dyg, pref, rhs = W.make_xglobal_inputs(wl, cuda_device)
    h = gene_nlx_create(wl.nx, wl.nky0, wl.planes)
    try:
        with pytest.raises(GeneNLError):
            gene_nlx_compute(h, vex, vey, dxg, rhs, pref, rhs, 1.0)     # rhs overlaps an input
        with pytest.raises(GeneNLError):
            gene_nlx_compute(h, vex, vey, dxg, dyg, pref, 0, 1.0)       # NULL
        gene_nlx_compute(h, vex, vey, dxg, dyg, pref, rhs, 1.0)
        torch.cuda.synchronize()
    finally:
        gene_nlx_destroy(h)
