"""Shared helpers of the parity tests: run the CUDA path through the C ABI, run the oracle on sampled
planes, and the error metric of SURVEY.md 8(c) R14 / BASELINE.json north_star:
    err_p = || rhs_gpu_p - rhs_ref_p ||_2 / || scale * N_ref_p ||_2 ,  max over planes <= 1e-11."""
import numpy as np
import torch

import oracle
from paper_1310_1485_b200 import workloads as W

TOL = 1e-11  # north_star: max over planes of ||N_gpu - N_ref||_2 / ||N_ref||_2 <= 1e-11


def sample_planes(wl, n, seed=0):
    """Planes to compare when the oracle cannot do them all.  Never truncated: always planes 0 and P-1 and the 16
    corners (first/last index of each of z, v, w, s: both species, first and last slab), then one seeded random plane in
    EVERY (w,s) slab (a wrong plane -> CTA map or a ragged batch tail shows up inside slabs, not only at the ends), then
    seeded random planes until at least max(n, corners + slabs + 32) planes are picked."""
    P = wl.planes
    picks = {0, P - 1}
    for z in (0, wl.nz - 1):
        for v in (0, wl.nv - 1):
            for w in (0, wl.nw - 1):
                for s in (0, wl.nspec - 1):
                    picks.add(z + wl.nz * (v + wl.nv * (w + wl.nw * s)))
    rng = np.random.default_rng(seed)
    per_slab = wl.nz * wl.nv
    for ws in range(wl.nw * wl.nspec):
        picks.add(ws * per_slab + int(rng.integers(0, per_slab)))
    want = min(P, max(n, len(picks) + 32))
    while len(picks) < want:
        picks.add(int(rng.integers(0, P)))
    return np.array(sorted(picks))


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


def plane_max_errors(wl, out_planes, ref, R_in):
    """Element-wise companion of the R14 norm: per plane max |rhs_gpu - rhs_ref| / max |scale N_ref|.  The L2 norm over
    a 65 536-mode plane hides one wrong mode at 1e-9; this bound (same 1e-11) does not."""
    num = np.abs(out_planes - ref).reshape(len(ref), -1).max(axis=1)
    den = np.abs(ref - R_in).reshape(len(ref), -1).max(axis=1)
    assert np.all(den > 0)
    return num / den


def gpu_compute(wl, chi, g, rhs, scale=None, host=False, scratch_bytes=None, plane_kernel=None):
    """rhs += scale*N through the C ABI; returns the updated rhs tensor (a new tensor)."""
    from paper_1310_1485_b200 import GeneNL
    out = rhs.clone()
    with GeneNL(wl, scratch_bytes=scratch_bytes, plane_kernel=plane_kernel) as nl:
        if host:
            nl.compute_host(chi, g, out, scale)
        else:
            nl.compute(chi, g, out, scale)
            torch.cuda.synchronize()
    return out


def check_parity(wl, device, nsample=None, host=False, tol=TOL, backend=oracle.DFT_RECURSIVE, scratch_bytes=None,
                 plane_kernel=None):
    chi, g, rhs = W.make_inputs(wl, device if not host else "cpu")
    if host:
        chi, g, rhs = chi.pin_memory(), g.pin_memory(), rhs.pin_memory()
    out = gpu_compute(wl, chi, g, rhs, host=host, scratch_bytes=scratch_bytes, plane_kernel=plane_kernel)
    planes = np.arange(wl.planes) if nsample is None or nsample >= wl.planes else sample_planes(wl, nsample, wl.seed)
    err, emax = [], []
    for c0 in range(0, len(planes), 1024):   # the oracle in bounded chunks (host memory)
        sel = planes[c0:c0 + 1024]
        ref, R, _, _ = oracle_on_planes(wl, chi, g, rhs, sel, backend=backend)
        idx = torch.as_tensor(sel, dtype=torch.long, device=out.device)
        got = W.as_planes(out, wl)[idx].cpu().numpy()
        err.append(plane_errors(wl, got, ref, R))
        emax.append(plane_max_errors(wl, got, ref, R))
    err, emax = np.concatenate(err), np.concatenate(emax)
    assert err.max() <= tol, f"{wl.name}: max plane error {err.max():.3e} at plane {planes[err.argmax()]}"
    assert emax.max() <= tol, f"{wl.name}: max element error {emax.max():.3e} at plane {planes[emax.argmax()]}"
    # Nyquist row of rhs untouched, bit for bit (R6)
    h = wl.nx0 // 2
    assert torch.equal(W.as_planes(out, wl)[:, :, h], W.as_planes(rhs, wl)[:, :, h])
    return err.max()
