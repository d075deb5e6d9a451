"""Shared helpers of the parity tests: run the CUDA path through the C ABI, run the oracle on sampled
planes, and the error metric of SURVEY.md 8(c) R14 / BASELINE.json north_star:
    err_p = || rhs_gpu_p - rhs_ref_p ||_2 / || scale * N_ref_p ||_2 ,  max over planes <= 1e-11."""
import numpy as np
import torch

import oracle
from paper_1310_1485_b200 import workloads as W

TOL = 1e-11  # north_star: max over planes of ||N_gpu - N_ref||_2 / ||N_ref||_2 <= 1e-11


def sample_planes(wl, n, seed=0):
    """First/last plane, first/last index of each of z, v, w, s, plus seeded random planes."""
    P = wl.planes
    picks = {0, P - 1}
    for z in (0, wl.nz - 1):
        for v in (0, wl.nv - 1):
            for w in (0, wl.nw - 1):
                for s in (0, wl.nspec - 1):
                    picks.add(z + wl.nz * (v + wl.nv * (w + wl.nw * s)))
    rng = np.random.default_rng(seed)
    while len(picks) < min(n, P):
        picks.add(int(rng.integers(0, P)))
    return np.array(sorted(picks)[:max(n, 2)] if len(picks) > n else sorted(picks))


def oracle_on_planes(wl, chi, g, rhs_in, planes, scale=None, backend=oracle.DFT_RECURSIVE):
    """Oracle result for the selected planes; inputs are torch tensors on any device."""
    scale = wl.scale if scale is None else scale
    idx = torch.as_tensor(planes, dtype=torch.long, device=g.device)
    cidx = torch.as_tensor([W.chi_plane_of(wl, int(p)) for p in planes], dtype=torch.long, device=g.device)
    G = W.as_planes(g, wl)[idx].cpu().numpy()
    X = W.as_planes(chi, wl)[cidx].cpu().numpy()
    R = W.as_planes(rhs_in, wl)[idx].cpu().numpy()
    ref = oracle.nl_pseudospectral(X, G, R, scale, wl.kxmin, wl.kymin, backend=backend)
    return ref, R, X, G


def plane_errors(wl, out_planes, ref, R_in):
    """R14 error per plane; out_planes, ref, R_in: (n, nky0, nx0) numpy."""
    num = np.linalg.norm((out_planes - ref).reshape(len(ref), -1), axis=1)
    den = np.linalg.norm((ref - R_in).reshape(len(ref), -1), axis=1)
    assert np.all(den > 0)
    return num / den


def gpu_compute(wl, chi, g, rhs, scale=None, host=False):
    """rhs += scale*N through the C ABI; returns the updated rhs tensor (a new tensor)."""
    from paper_1310_1485_b200 import GeneNL
    out = rhs.clone()
    with GeneNL(wl) as nl:
        if host:
            nl.compute_host(chi, g, out, scale)
        else:
            nl.compute(chi, g, out, scale)
            torch.cuda.synchronize()
    return out


def check_parity(wl, device, nsample=None, host=False, tol=TOL, backend=oracle.DFT_RECURSIVE):
    chi, g, rhs = W.make_inputs(wl, device if not host else "cpu")
    if host:
        chi, g, rhs = chi.pin_memory(), g.pin_memory(), rhs.pin_memory()
    out = gpu_compute(wl, chi, g, rhs, host=host)
    planes = np.arange(wl.planes) if nsample is None or nsample >= wl.planes else sample_planes(wl, nsample, wl.seed)
    ref, R, _, _ = oracle_on_planes(wl, chi, g, rhs, planes, backend=backend)
    idx = torch.as_tensor(planes, dtype=torch.long, device=out.device)
    got = W.as_planes(out, wl)[idx].cpu().numpy()
    err = plane_errors(wl, got, ref, R)
    assert err.max() <= tol, f"{wl.name}: max plane error {err.max():.3e} at plane {planes[err.argmax()]}"
    # Nyquist row of rhs untouched, bit for bit (R6)
    h = wl.nx0 // 2
    assert torch.equal(W.as_planes(out, wl)[:, :, h], W.as_planes(rhs, wl)[:, :, h])
    return err.max()
