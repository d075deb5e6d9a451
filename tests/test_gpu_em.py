"""Electromagnetic case with chi composed on the device (gene_nl_compute_em): parity against
the CPU oracle fed with chi_p = phi_bar - vpar * apar_bar composed per plane in numpy (FP64), and agreement with the
per-plane-chi path of the library (chi_has_v = 1) on the same data."""
import numpy as np
import pytest
import torch

import oracle
from helpers import TOL, plane_errors
from paper_1310_1485_b200 import workloads as W

pytestmark = pytest.mark.gpu


def em_inputs(wl, device):
    """phi_bar, apar_bar (chi layout without v), vpar (nv*nspec), g, rhs from the workload's seeded generator."""
    assert not wl.chi_has_v
    phi, g, rhs = W.make_inputs(wl, device)
    wl2 = W.Workload(wl.name + "_apar", wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, False,
                     wl.seed + 77, wl.rhs_random, wl.scale)
    apar, _, _ = W.make_inputs(wl2, device)
    v = np.linspace(-3.0, 3.0, wl.nv)
    vpar = np.concatenate([v * (1.0 + 0.5 * s) for s in range(wl.nspec)])   # species-dependent thermal velocity
    return phi, apar, vpar, g, rhs


def composed_chi(wl, phi, apar, vpar):
    """(planes, nky0, nx0) numpy: chi_p = phi_q - vpar[v + nv s] apar_q, p = z + nz (v + nv (w + nw s))."""
    X, A = (W.as_planes(t, wl).cpu().numpy() for t in (phi, apar))
    chi = np.empty((wl.planes, wl.nky0, wl.nx0), complex)
    for p in range(wl.planes):
        z, v = p % wl.nz, (p // wl.nz) % wl.nv
        ws = p // (wl.nz * wl.nv)
        s = ws // wl.nw
        q = z + wl.nz * ws
        chi[p] = X[q] - vpar[v + wl.nv * s] * A[q]
    return chi


def run_em(wl, phi, apar, vpar, g, rhs, scratch_bytes=None, host=False, plane_kernel=None):
    from paper_1310_1485_b200 import (GENE_NL_CHI_EM, gene_nl_compute_em, gene_nl_compute_em_host, gene_nl_create,
                                      gene_nl_destroy, gene_nl_set_plane_kernel, gene_nl_set_scratch_bytes)
    out = rhs.clone()
    h = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, GENE_NL_CHI_EM)
    try:
        if plane_kernel is not None:
            gene_nl_set_plane_kernel(h, plane_kernel)
        if scratch_bytes is not None:
            gene_nl_set_scratch_bytes(h, scratch_bytes)
        if host:
            hp, ha, hg, ho = (t.cpu().pin_memory() for t in (phi, apar, g, out))
            gene_nl_compute_em_host(h, hp, ha, vpar, hg, ho, wl.scale)
            out = ho.to(rhs.device)
        else:
            gene_nl_compute_em(h, phi, apar, vpar, g, out, wl.scale)
            gene_nl_compute_em(h, phi, apar, 0.0 * vpar, g, out, 0.0)   # a second call reuses the v_par staging buffer
            torch.cuda.synchronize()
    finally:
        gene_nl_destroy(h)
    return out


SHAPES = [(16, 8, 3, 5, 2, 2), (64, 32, 2, 3, 2, 1), (96, 48, 2, 4, 1, 2), (96, 48, 3, 5, 3, 2), (128, 32, 3, 3, 1, 1),
          (96, 48, 8, 10, 2, 2),    # 320 planes > 2 x 148 groups of one CTA: every group walks on to a second and third
                                    # plane, and v_par's species index changes inside a group's walk
          (256, 64, 4, 5, 3, 2),    # 120 planes > 3 x 37 groups of four CTAs
          (256, 64, 2, 2, 1, 2), (256, 64, 2, 3, 3, 2),
          (32, 128, 1, 3, 1, 1),
          (256, 64, 36, 2, 1, 1)]   # chi rows of a chunk beyond 40 MB: k_ybracket<EM> walks its tiles v-fastest


# the composition runs in the group kernel where one exists (144 x 144 and 384 x 192 planes), else in k_ybracket<EM>;
# kind 3 = GENE_NL_KERNEL_BATCHED forces the latter everywhere
@pytest.mark.parametrize("kind", [None, 3])
@pytest.mark.parametrize("nx0,nky0,nz,nv,nw,nspec", SHAPES)
def test_em_matches_oracle_on_composed_chi(cuda_device, nx0, nky0, nz, nv, nw, nspec, kind):
    wl = W.small_workload(nx0, nky0, nz, nv, nw, nspec, 0.03, 0.07, False, seed=200 + nx0 + nky0)
    phi, apar, vpar, g, rhs = em_inputs(wl, cuda_device)
    out = run_em(wl, phi, apar, vpar, g, rhs, plane_kernel=kind)
    chi = composed_chi(wl, phi, apar, vpar)
    G, R = (W.as_planes(t, wl).cpu().numpy() for t in (g, rhs))
    ref = oracle.nl_pseudospectral(chi, G, R, wl.scale, wl.kxmin, wl.kymin)
    assert plane_errors(wl, W.as_planes(out, wl).cpu().numpy(), ref, R).max() <= TOL


def test_em_under_a_tiny_scratch_budget_and_against_the_per_plane_chi_path(cuda_device):
    from helpers import gpu_compute
    wl = W.small_workload(64, 32, 5, 7, 2, 2, 0.05, 0.05, False, seed=31)
    phi, apar, vpar, g, rhs = em_inputs(wl, cuda_device)
    out = run_em(wl, phi, apar, vpar, g, rhs, scratch_bytes=2 << 20)
    chi = composed_chi(wl, phi, apar, vpar)
    G, R = (W.as_planes(t, wl).cpu().numpy() for t in (g, rhs))
    ref = oracle.nl_pseudospectral(chi, G, R, wl.scale, wl.kxmin, wl.kymin)
    assert plane_errors(wl, W.as_planes(out, wl).cpu().numpy(), ref, R).max() <= TOL
    # the library's own per-plane-chi path on the composed chi
    wlv = W.small_workload(64, 32, 5, 7, 2, 2, 0.05, 0.05, True, seed=31)
    chi_t = torch.from_numpy(chi).to(cuda_device).view(wlv.chi_shape)
    out_v = gpu_compute(wlv, chi_t, g, rhs)
    d = (out - out_v).abs().max().item()
    assert d <= 1e-12 * (out_v - rhs).abs().max().item()


def test_em_host_entry_point_matches_the_device_entry_point(cuda_device):
    """gene_nl_compute_em_host streams (w,s) slabs through the same kernels: the same bits as gene_nl_compute_em; the
    species index of a slab (v_par is per species) must survive the slab-by-slab walk."""
    for nx0, nky0 in ((64, 32), (96, 48)):     # batched kernels / group kernel behind the streaming driver
        wl = W.small_workload(nx0, nky0, 3, 4, 3, 2, 0.05, 0.05, False, seed=33)
        phi, apar, vpar, g, rhs = em_inputs(wl, cuda_device)
        dev = run_em(wl, phi, apar, vpar, g, rhs)
        hst = run_em(wl, phi, apar, vpar, g, rhs, host=True)
        assert torch.equal(dev, hst)
        chi = composed_chi(wl, phi, apar, vpar)
        G, R = (W.as_planes(t, wl).cpu().numpy() for t in (g, rhs))
        ref = oracle.nl_pseudospectral(chi, G, R, wl.scale, wl.kxmin, wl.kymin)
        assert plane_errors(wl, W.as_planes(hst, wl).cpu().numpy(), ref, R).max() <= TOL


def test_em_full_size_config4_grid_sampled_planes(cuda_device):
    """The run BASELINE.md quotes (bench.py --em): configs[4]'s grid, 73 728 planes, phi_bar and A_par_bar supplied and chi
    composed in the group kernel; >= 160 sampled planes (both ends, every (w,s) slab) against the oracle on chi composed
    in numpy for those planes."""
    from helpers import plane_max_errors, sample_planes
    c4 = W.CONFIGS[4]
    wl = W.Workload("cfg4_em_composed", c4.nx0, c4.nky0, c4.nz, c4.nv, c4.nw, c4.nspec, c4.kxmin, c4.kymin, False,
                    c4.seed, c4.rhs_random, c4.scale)
    need = 16 * wl.nx0 * wl.nky0 * 3.3 * wl.planes
    torch.cuda.empty_cache()
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip(f"{wl.name} needs {need / 2**30:.0f} GiB of device memory")
    phi, apar, vpar, g, rhs = em_inputs(wl, cuda_device)
    out = run_em(wl, phi, apar, vpar, g, rhs)
    planes = sample_planes(wl, 160, wl.seed)
    X, A = (W.as_planes(t, wl) for t in (phi, apar))
    chi = np.empty((len(planes), wl.nky0, wl.nx0), complex)
    for i, p in enumerate(planes):
        p = int(p)
        z, v, ws = p % wl.nz, (p // wl.nz) % wl.nv, p // (wl.nz * wl.nv)
        q = z + wl.nz * ws
        chi[i] = X[q].cpu().numpy() - vpar[v + wl.nv * (ws // wl.nw)] * A[q].cpu().numpy()
    idx = torch.as_tensor(planes, dtype=torch.long, device=g.device)
    G, R, got = (W.as_planes(t, wl)[idx].cpu().numpy() for t in (g, rhs, out))
    ref = oracle.nl_pseudospectral(chi, G, R, wl.scale, wl.kxmin, wl.kymin)
    assert plane_errors(wl, got, ref, R).max() <= TOL
    assert plane_max_errors(wl, got, ref, R).max() <= TOL
    h = wl.nx0 // 2
    assert torch.equal(W.as_planes(out, wl)[:, :, h], W.as_planes(rhs, wl)[:, :, h])


def test_em_refuses_stream_capture_and_leaves_the_capture_intact(cuda_device):
    """gene_nl_compute_em stages v_par through a pinned host buffer and waits on the host for the previous copy, which a
    capturing stream does not allow: the call says so (GENE_NL_EUNSUPPORTED) instead of breaking the caller's capture."""
    from paper_1310_1485_b200 import GENE_NL_CHI_EM, GeneNLError, gene_nl_compute_em, gene_nl_create, gene_nl_destroy
    wl = W.small_workload(96, 48, 2, 2, 1, 1, 0.1, 0.1, False, seed=9)
    phi, apar, vpar, g, rhs = em_inputs(wl, cuda_device)
    out = rhs.clone()
    h = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, GENE_NL_CHI_EM)
    try:
        gene_nl_compute_em(h, phi, apar, vpar, g, out, wl.scale)
        torch.cuda.synchronize()
        expect = out.clone()
        x = torch.zeros(8, device=cuda_device)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            with pytest.raises(GeneNLError, match="captured"):
                gene_nl_compute_em(h, phi, apar, vpar, g, out, wl.scale)
            x.add_(1.0)
        graph.replay()
        torch.cuda.synchronize()
        assert x.eq(1.0).all() and torch.equal(out, expect)
    finally:
        gene_nl_destroy(h)


def test_em_errors(cuda_device):
    from paper_1310_1485_b200 import (GENE_NL_CHI_EM, GeneNLError, gene_nl_compute, gene_nl_compute_em, gene_nl_create,
                                      gene_nl_destroy)
    wl = W.small_workload(32, 16, 2, 2, 1, 1, 0.1, 0.1, False, seed=8)
    phi, apar, vpar, g, rhs = em_inputs(wl, cuda_device)
    h_em = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, GENE_NL_CHI_EM)
    h = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, 0)
    try:
        with pytest.raises(GeneNLError):
            gene_nl_compute(h_em, phi, g, rhs, 1.0)            # an EM plan takes gene_nl_compute_em only
        with pytest.raises(GeneNLError):
            gene_nl_compute_em(h, phi, apar, vpar, g, rhs, 1.0)  # and the reverse
        with pytest.raises(GeneNLError):
            gene_nl_compute_em(h_em, phi, apar, vpar, g, g, 1.0)  # rhs overlaps g
    finally:
        gene_nl_destroy(h_em)
        gene_nl_destroy(h)
