"""Seeded synthetic inputs for the ExB nonlinearity: the five workloads of BASELINE.json `configs`.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests, and therefore
holds none of the method's arithmetic (no derivative, transform, bracket or accumulation): only the
grid sizes, the wavenumber grid needed by the input recipe, and the random fill.

Recipe (BASELINE.json configs[0], readings R6/R9/R10 of SURVEY.md sect. 8(c)); the data stand in for
GENE turbulence spectra (the paper's own workload is 64x16x24x96x16 double-complex):
  * g[kx,ky,z,v,w,s], kx fastest, complex128; chi[kx,ky,z,w,s] (no v) or, with chi_has_v, like g.
    As torch tensors (row-major): g (nspec,nw,nv,nz,nky0,nx0), chi (nspec,nw,nz,nky0,nx0).
  * value = (a+ib)/(1+(kx^2+ky^2)/0.25), a,b ~ N(0,1) from torch's seeded generator on the device
    the arrays are created on (Philox on CUDA).  The same bytes are fed to the CUDA path and to the
    oracle, so parity never depends on reproducing a random stream across devices (R10).
  * ky=0 column Hermitian: F[nx0-i,0] = conj F[i,0], F[0,0] real.  Nyquist row i = nx0/2 zeroed.
  * rhs: zeros (config 0) or a+ib without fall-off, Hermitian-consistent, Nyquist row zero (R9).
"""
from __future__ import annotations

from dataclasses import dataclass

import torch


@dataclass(frozen=True)
class Workload:
    name: str
    nx0: int
    nky0: int
    nz: int
    nv: int
    nw: int
    nspec: int
    kxmin: float
    kymin: float
    chi_has_v: bool
    seed: int
    rhs_random: bool
    scale: float

    @property
    def planes(self) -> int:
        return self.nz * self.nv * self.nw * self.nspec

    @property
    def chi_planes(self) -> int:
        return self.planes if self.chi_has_v else self.nz * self.nw * self.nspec

    @property
    def Nx(self) -> int:
        return 3 * self.nx0 // 2

    @property
    def Ny(self) -> int:
        return 3 * self.nky0

    @property
    def g_shape(self):
        return (self.nspec, self.nw, self.nv, self.nz, self.nky0, self.nx0)

    @property
    def chi_shape(self):
        if self.chi_has_v:
            return self.g_shape
        return (self.nspec, self.nw, self.nz, self.nky0, self.nx0)

    @property
    def plane_bytes(self) -> int:
        return 16 * self.nx0 * self.nky0


# BASELINE.json configs[0..4]
CONFIGS = (
    Workload("cfg0_tiny_16x8", 16, 8, 4, 4, 2, 1, 0.1, 0.1, False, 1, False, 1.0),
    Workload("cfg1_medium_128x32", 128, 32, 16, 32, 8, 2, 0.05, 0.05, False, 2, True, 0.7),
    Workload("cfg2_large_256x64", 256, 64, 16, 32, 8, 2, 0.025, 0.05, False, 3, True, 0.7),
    Workload("cfg3_hbm_512x128", 512, 128, 24, 32, 16, 2, 0.0125, 0.025, False, 4, True, 0.7),
    Workload("cfg4_em_96x48", 96, 48, 32, 48, 16, 3, 0.04, 0.04, True, 5, True, 0.7),
)


def small_workload(nx0=16, nky0=8, nz=2, nv=3, nw=2, nspec=1, kxmin=0.1, kymin=0.1,
                   chi_has_v=False, seed=11, rhs_random=True, scale=0.7, name=None) -> Workload:
    """A configs[0]-style workload of arbitrary (small) size, for parity cases and ragged tails."""
    name = name or f"small_{nx0}x{nky0}_{nz}.{nv}.{nw}.{nspec}_{'v' if chi_has_v else 'nov'}"
    return Workload(name, nx0, nky0, nz, nv, nw, nspec, kxmin, kymin, chi_has_v, seed, rhs_random, scale)


def kx_grid(wl: Workload, device="cpu") -> torch.Tensor:
    """kx of stored row i: kxmin*i below the Nyquist row, kxmin*(i-nx0) above it, 0 on it."""
    i = torch.arange(wl.nx0, device=device, dtype=torch.float64)
    kx = torch.where(i < wl.nx0 // 2, i, i - wl.nx0) * wl.kxmin
    kx[wl.nx0 // 2] = 0.0
    return kx


def ky_grid(wl: Workload, device="cpu") -> torch.Tensor:
    return torch.arange(wl.nky0, device=device, dtype=torch.float64) * wl.kymin


def _fill(shape, gen, device, falloff, wl: Workload, max_chunk_bytes=1 << 30) -> torch.Tensor:
    """complex128 tensor of `shape` (..., nky0, nx0) with the recipe above, made in bounded chunks."""
    out = torch.empty(shape, dtype=torch.complex128, device=device)
    flat = out.view(-1, wl.nky0, wl.nx0)
    per_plane = 16 * wl.nky0 * wl.nx0
    step = max(1, max_chunk_bytes // per_plane)
    damp = None
    if falloff:
        k2 = kx_grid(wl, device)[None, :] ** 2 + ky_grid(wl, device)[:, None] ** 2
        damp = 1.0 / (1.0 + k2 / 0.25)
    h = wl.nx0 // 2
    for p0 in range(0, flat.shape[0], step):
        blk = flat[p0:p0 + step]
        ab = torch.randn(blk.shape + (2,), dtype=torch.float64, device=device, generator=gen)
        blk.copy_(torch.view_as_complex(ab))
        del ab
        if damp is not None:
            blk.mul_(damp)
        # ky = 0 column Hermitian in kx, (0,0) real; Nyquist row zero
        blk[:, 0, h + 1:] = torch.conj(torch.flip(blk[:, 0, 1:h], dims=[1]))
        blk[:, 0, 0] = blk[:, 0, 0].real.to(torch.complex128)
        blk[:, :, h] = 0
    return out


def make_inputs(wl: Workload, device="cpu"):
    """(chi, g, rhs) for a workload, created on `device` from the workload's seed."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(wl.seed)
    g = _fill(wl.g_shape, gen, dev, True, wl)
    chi = _fill(wl.chi_shape, gen, dev, True, wl)
    if wl.rhs_random:
        rhs = _fill(wl.g_shape, gen, dev, False, wl)
    else:
        rhs = torch.zeros(wl.g_shape, dtype=torch.complex128, device=dev)
    return chi, g, rhs


def chi_plane_of(wl: Workload, p):
    """Index of the chi plane used by g plane p (p = z + nz*(v + nv*(w + nw*s)))."""
    if wl.chi_has_v:
        return p
    z = p % wl.nz
    ws = p // (wl.nz * wl.nv)
    return z + wl.nz * ws


def as_planes(t: torch.Tensor, wl: Workload) -> torch.Tensor:
    """View an array as (planes, nky0, nx0)."""
    return t.view(-1, wl.nky0, wl.nx0)


def shard_slabs(wl: Workload, rank: int, world: int):
    """Contiguous range [s0, s1) of the nw*nspec (w,s) slabs owned by `rank`: g, rhs AND
    chi shard together along the slowest indices, so the bracket needs no exchange between ranks."""
    nslab = wl.nw * wl.nspec
    base, extra = divmod(nslab, world)
    s0 = rank * base + min(rank, extra)
    return s0, s0 + base + (1 if rank < extra else 0)


def shard_arrays(wl: Workload, chi, g, rhs, rank: int, world: int):
    """(sub-workload, chi, g, rhs views) of one rank's slabs; the sub-workload has nw = slabs, nspec = 1."""
    s0, s1 = shard_slabs(wl, rank, world)
    n = s1 - s0
    sub = Workload(f"{wl.name}_rank{rank}of{world}", wl.nx0, wl.nky0, wl.nz, wl.nv, max(n, 0), 1,
                   wl.kxmin, wl.kymin, wl.chi_has_v, wl.seed, wl.rhs_random, wl.scale)
    gs = g.reshape((wl.nw * wl.nspec,) + wl.g_shape[2:])[s0:s1]
    rs = rhs.reshape((wl.nw * wl.nspec,) + wl.g_shape[2:])[s0:s1]
    cs = chi.reshape((wl.nw * wl.nspec,) + wl.chi_shape[2:])[s0:s1]
    return sub, cs, gs, rs


# ---------------------------------------------------------------------------------------------------------
# x-global variant: the paper's own workload, 64 x 16 planes ("64 x 16 x 24 x 96
# x 16" grid points in x, ky, z, v, mu), timed over 589 824 planes device-resident (Table 4).
# Recipe: five arrays (planes, nky0, nx) complex128, x fastest.  Inputs a+ib ~ N(0,1) with a fall-off 1/(1+(j/4)^2)
# in the ky index and a smooth envelope in x; the ky = 0 row is real (the fields are real).  rhs ~ N(0,1), ky = 0 row
# real.  pref[x] = 1 + 0.5*cos(2 pi x/nx) (an x-dependent prefactor), scale = 0.7.  Stands in for GENE data.
# ---------------------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class XGlobalWorkload:
    name: str
    nx: int
    nky0: int
    planes: int
    seed: int
    scale: float

    @property
    def Ny(self) -> int:
        return 3 * self.nky0

    @property
    def shape(self):
        return (self.planes, self.nky0, self.nx)

    @property
    def plane_bytes(self) -> int:
        return 16 * self.nx * self.nky0


XGLOBAL_PAPER = XGlobalWorkload("xglobal_paper_64x16_589824", 64, 16, 589824, 6, 0.7)
XGLOBAL_SMALL = XGlobalWorkload("xglobal_small_64x16_4096", 64, 16, 4096, 7, 0.7)


def make_xglobal_inputs(wl: XGlobalWorkload, device="cpu", max_chunk_bytes=1 << 30):
    """(vex, vey, dxg, dyg, pref, rhs) created on `device` from the workload's seed."""
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(wl.seed)
    j = torch.arange(wl.nky0, device=dev, dtype=torch.float64)
    x = torch.arange(wl.nx, device=dev, dtype=torch.float64)
    damp = (1.0 / (1.0 + (j / 4.0) ** 2))[:, None] * (0.75 + 0.25 * torch.sin(2 * torch.pi * (x + 0.5) / wl.nx))[None, :]
    step = max(1, max_chunk_bytes // wl.plane_bytes)

    def fill(falloff):
        out = torch.empty(wl.shape, dtype=torch.complex128, device=dev)
        for p0 in range(0, wl.planes, step):
            blk = out[p0:p0 + step]
            ab = torch.randn(blk.shape + (2,), dtype=torch.float64, device=dev, generator=gen)
            blk.copy_(torch.view_as_complex(ab))
            del ab
            if falloff:
                blk.mul_(damp)
            blk[:, 0, :] = blk[:, 0, :].real.to(torch.complex128)
        return out

    vex, vey, dxg, dyg = (fill(True) for _ in range(4))
    rhs = fill(False)
    pref = 1.0 + 0.5 * torch.cos(2 * torch.pi * x / wl.nx)
    return vex, vey, dxg, dyg, pref, rhs
