"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on the same
seeded inputs (north_star: max over planes of ||N_gpu - N_ref||_2/||N_ref||_2 <= 1e-11)."""
import os

import numpy as np
import pytest
import torch

import oracle
from helpers import TOL, check_parity, gpu_compute, oracle_on_planes, plane_errors, sample_planes
from paper_1310_1485_b200 import workloads as W

pytestmark = pytest.mark.gpu


def test_config0_all_planes_against_oracle_and_definition(cuda_device):
    wl = W.CONFIGS[0]
    err = check_parity(wl, cuda_device, backend=oracle.DFT_NAIVE)
    assert err <= TOL
    # and directly against the definition (truncated convolution) on every plane
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    out = W.as_planes(gpu_compute(wl, chi, g, rhs), wl).cpu().numpy()
    X, G = W.as_planes(chi, wl).cpu().numpy(), W.as_planes(g, wl).cpu().numpy()
    for p in range(wl.planes):
        N = oracle.nl_convolution_plane(X[W.chi_plane_of(wl, p)], G[p], wl.kxmin, wl.kymin)
        assert np.linalg.norm(out[p] - wl.scale * N) <= TOL * np.linalg.norm(N)


# every instantiated x length (nx0 = 2 Nx / 3) and y length (nky0 = Ny / 3), both chi layouts,
# extents that do not divide the batch sizes (ragged z / v tails once the budget is squeezed)
SHAPES = [
    (16, 8, 3, 5, 2, 1, False), (16, 8, 2, 3, 1, 2, True),
    (32, 16, 3, 2, 1, 1, False), (64, 32, 2, 3, 1, 1, True),
    (96, 48, 2, 2, 1, 1, True), (96, 48, 3, 2, 1, 1, False),
    (128, 32, 3, 3, 1, 1, False), (128, 64, 1, 2, 1, 1, True),
    (256, 64, 2, 2, 1, 1, False), (32, 128, 1, 3, 1, 1, False),
    (512, 16, 1, 2, 1, 1, True), (16, 8, 1, 1, 1, 1, False),
    (256, 64, 36, 2, 1, 1, False),   # 384 x 192: the group kernel by default (the batched kernels of this shape,
                                     # k_xinv_p<ZT> + k_ybracket_t with its v-fastest tile walk, run under kind 3 in
                                     # test_spread_kernels_small_shapes_all_planes)
    # Nx = 768 with chi shared over v and Ny <= 192: k_xinv_p<768,...,ZT> + k_ybracket_t (on by default at these sizes)
    (512, 16, 2, 3, 1, 1, False), (512, 64, 1, 2, 1, 1, False),
    (512, 128, 1, 2, 1, 1, False),   # the plane shape of configs[3]: the group kernel (G = 8) by default; the batched kernels of
                                     # this shape run in test_768x384_kernel_families
    (512, 128, 1, 1, 1, 1, True),    # chi per plane at 768 x 384: batched (k_xinv<768,...,SEQ> + k_ybracket_cv<384> + k_xfwd<768>)
    # the wider size list (2^a 3^b): Nx = 288, 576, 1152, 1536 and Ny = 288, 576 (batched kernels)
    (192, 32, 2, 3, 1, 1, False), (192, 96, 1, 2, 1, 1, True),     # 288 x 96 (transposed-Z path), 288 x 288
    (384, 96, 1, 2, 1, 1, False), (32, 192, 2, 2, 1, 1, False),    # 576 x 288, 48 x 576
    (768, 16, 1, 2, 1, 1, True), (1024, 16, 1, 3, 1, 1, False),    # 1152 x 48, 1536 x 48
    (1024, 64, 1, 1, 1, 1, False),                                 # 1536 x 192: 64 Ki modes per plane
]


@pytest.mark.parametrize("nx0,nky0,nz,nv,nw,nspec,chi_has_v", SHAPES)
def test_small_shapes_all_planes(cuda_device, nx0, nky0, nz, nv, nw, nspec, chi_has_v):
    wl = W.small_workload(nx0, nky0, nz, nv, nw, nspec, 0.03, 0.07, chi_has_v, seed=nx0 + nky0)
    check_parity(wl, cuda_device)


@pytest.mark.parametrize("budget_mb", [1, 3])
def test_ragged_batches_under_a_tiny_scratch_budget(cuda_device, budget_mb):
    """gene_nl_set_scratch_bytes: more and smaller batches (ragged z and v tails), never a different result.
    64 x 32 planes take the fused kernel (the budget bounds its chi cache: several launches), 64 x 64 the batched ones."""
    for nky0 in (32, 64):
        for chi_has_v in (False, True):
            wl = W.small_workload(64, nky0, 5, 7, 2, 1, 0.05, 0.05, chi_has_v, seed=21)
            check_parity(wl, cuda_device, scratch_bytes=budget_mb << 20)


def test_set_scratch_bytes_changes_the_batching_not_the_bits(cuda_device):
    from paper_1310_1485_b200 import GeneNL, GeneNLError, gene_nl_set_scratch_bytes
    wl = W.small_workload(64, 64, 5, 7, 2, 1, 0.05, 0.05, False, seed=23)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    base = gpu_compute(wl, chi, g, rhs)
    with GeneNL(wl) as nl:
        n0 = nl.launches_per_compute
        gene_nl_set_scratch_bytes(nl.h, 2 << 20)
        assert nl.launches_per_compute > n0
        out = rhs.clone()
        nl.compute(chi, g, out)
        torch.cuda.synchronize()
        assert torch.equal(out, base)                 # planes are independent: the same bits whatever the batching
        with pytest.raises(GeneNLError):
            gene_nl_set_scratch_bytes(nl.h, 1000)      # below 1 MiB
        nl.compute(chi, g, out)                        # the plan still works afterwards
        torch.cuda.synchronize()


def test_properties_scale_zero_linearity_antisymmetry(cuda_device):
    wl = W.small_workload(64, 32, 2, 3, 1, 1, 0.05, 0.05, True, seed=5)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    assert torch.equal(gpu_compute(wl, chi, g, rhs, scale=0.0), rhs)        # scale = 0: bit-identical
    zero = torch.zeros_like(rhs)
    n1 = gpu_compute(wl, chi, g, zero, scale=1.0)
    n2 = gpu_compute(wl, chi, g, zero, scale=-2.5)
    assert (n2 + 2.5 * n1).abs().max() <= 1e-14 * n1.abs().max()             # linear in scale
    nswap = gpu_compute(wl, g, chi, zero, scale=1.0)                        # N(g,chi) = -N(chi,g)
    assert (n1 + nswap).abs().max() <= 1e-13 * n1.abs().max()
    nself = gpu_compute(wl, g, g, zero, scale=1.0)                          # N(g,g) = 0
    assert nself.abs().max() <= 1e-13 * n1.abs().max()
    # deterministic: two runs give the same bits
    assert torch.equal(n1, gpu_compute(wl, chi, g, zero, scale=1.0))


def test_nyquist_rows_of_inputs_are_ignored(cuda_device):
    wl = W.small_workload(32, 16, 2, 2, 1, 1, 0.1, 0.1, False, seed=6)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    base = gpu_compute(wl, chi, g, rhs)
    chi2, g2 = chi.clone(), g.clone()
    chi2[..., wl.nx0 // 2] = 5.0 + 1.0j
    g2[..., wl.nx0 // 2] = -2.0 + 7.0j
    assert torch.equal(gpu_compute(wl, chi2, g2, rhs), base)


def test_non_hermitian_ky0_column_follows_reading_R7(cuda_device):
    wl = W.small_workload(32, 16, 1, 2, 1, 1, 0.1, 0.1, True, seed=7)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    gen = torch.Generator(device=cuda_device).manual_seed(1)
    for t in (chi, g):
        col = torch.randn(t[..., 0, :].shape + (2,), dtype=torch.float64, device=cuda_device, generator=gen)
        t[..., 0, :] = torch.view_as_complex(col)
    out = gpu_compute(wl, chi, g, rhs)
    planes = np.arange(wl.planes)
    ref, R, _, _ = oracle_on_planes(wl, chi, g, rhs, planes, backend=oracle.DFT_NAIVE)
    assert plane_errors(wl, W.as_planes(out, wl).cpu().numpy(), ref, R).max() <= TOL


def test_host_entry_point_matches_oracle(cuda_device):
    check_parity(W.CONFIGS[0], cuda_device, host=True)
    for nky0 in (32, 64):           # fused and batched kernels behind the streaming driver
        for chi_has_v in (False, True):
            wl = W.small_workload(64, nky0, 5, 3, 2, 2, 0.05, 0.05, chi_has_v, seed=22)
            check_parity(wl, cuda_device, host=True, scratch_bytes=2 << 20)


def test_errors_are_reported_not_swallowed(cuda_device):
    from paper_1310_1485_b200 import GeneNL, GeneNLError, gene_nl_create
    with pytest.raises(GeneNLError):
        gene_nl_create(20, 8, 1, 1, 1, 1, 0.1, 0.1, 0)      # Nx = 30: no kernel
    with pytest.raises(GeneNLError):
        gene_nl_create(16, 7, 1, 1, 1, 1, 0.1, 0.1, 0)      # Ny = 21
    with pytest.raises(GeneNLError):
        gene_nl_create(15, 8, 1, 1, 1, 1, 0.1, 0.1, 0)      # odd nx0
    with pytest.raises(GeneNLError):
        gene_nl_create(16, 8, 0, 1, 1, 1, 0.1, 0.1, 0)      # empty extent
    wl = W.CONFIGS[0]
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    with GeneNL(wl) as nl:
        with pytest.raises(GeneNLError):
            nl.compute(chi, g, g)                             # rhs overlaps g
        with pytest.raises(GeneNLError):
            nl.compute(chi, g, rhs.data_ptr() + 8)            # misaligned
        with pytest.raises(GeneNLError):
            nl.compute(0, g, rhs)                             # NULL
        nl.compute(chi, g, rhs)                               # and the plan still works afterwards
        torch.cuda.synchronize()


def _full_size(cuda_device, idx, nsample, plane_kernel=None):
    wl = W.CONFIGS[idx]
    need = 16 * wl.nx0 * wl.nky0 * (3 * wl.planes + wl.chi_planes) * 1.15
    torch.cuda.empty_cache()       # blocks torch still caches from earlier tests are not "free" to the driver
    free, _ = torch.cuda.mem_get_info()
    if free < need:
        pytest.skip(f"{wl.name} needs {need / 2**30:.0f} GiB of device memory")
    return check_parity(wl, cuda_device, nsample=nsample, plane_kernel=plane_kernel)


def test_config1_full_size_all_planes(cuda_device):
    _full_size(cuda_device, 1, None)       # all 8192 planes (the oracle needs ~5 s on 16 cores)


def test_config2_full_size_all_planes(cuda_device):
    _full_size(cuda_device, 2, None)       # all 8192 planes (~25 s)


def test_config4_full_size_sampled_planes(cuda_device):
    _full_size(cuda_device, 4, 160)        # corners, one random plane in each of the 48 (w,s) slabs, random planes


def test_config3_full_size_sampled_planes(cuda_device):
    _full_size(cuda_device, 3, 96)         # corners, one random plane in each of the 32 (w,s) slabs, random planes


@pytest.mark.parametrize("world", [2, 3])
def test_plane_sharded_ranks_assemble_to_the_unsharded_result(cuda_device, world):
    """planes are independent given chi, so (w,s) slabs shard over ranks with no
    exchange.  One GPU here: each rank's shard (workloads.shard_arrays) goes through gene_nl_compute in turn and the
    assembled rhs must equal the unsharded call bit for bit; batched and fused kernels, chi with and without v."""
    for nx0, nky0, chi_has_v in ((64, 64, False), (128, 32, False), (64, 64, True)):
        wl = W.small_workload(nx0, nky0, 3, 4, 5, 1, 0.05, 0.05, chi_has_v, seed=50 + world)
        chi, g, rhs = W.make_inputs(wl, cuda_device)
        whole = gpu_compute(wl, chi, g, rhs)
        parts = []
        for rank in range(world):
            sub, cs, gs, rs = W.shard_arrays(wl, chi, g, rhs, rank, world)
            assert sub.nw >= 1
            parts.append(gpu_compute(sub, cs.contiguous(), gs.contiguous(), rs.contiguous()).reshape(-1))
        assert torch.equal(torch.cat(parts), whole.reshape(-1))


# ---- the kernels for planes beyond one SM that keep Z and P out of HBM (gene_nl_set_plane_kernel): 384 x 192 planes over a
# cluster of 8 CTAs with DSMEM hand-overs (1), or over a group of 4 co-resident CTAs with hand-overs through L2 (2) ----
SPREAD_SHAPES = [(256, 64, 1, 1, 1, 1),       # one plane: one cluster / group busy, the others idle
                 (256, 64, 2, 3, 1, 1),
                 (256, 64, 3, 5, 2, 2),       # 60 planes: several planes per cluster / group, chi shared by 5 planes
                 (256, 64, 36, 2, 1, 1)]
SPREAD_KINDS = [1, 2, 3, 4]                   # GENE_NL_KERNEL_CLUSTER, _GROUP (the default here), _BATCHED, _WARP


@pytest.mark.parametrize("kind", SPREAD_KINDS)
@pytest.mark.parametrize("nx0,nky0,nz,nv,nw,nspec", SPREAD_SHAPES)
def test_spread_kernels_small_shapes_all_planes(cuda_device, nx0, nky0, nz, nv, nw, nspec, kind):
    from paper_1310_1485_b200 import GeneNL
    wl = W.small_workload(nx0, nky0, nz, nv, nw, nspec, 0.03, 0.07, False, seed=300 + nz + nv)
    with GeneNL(wl, plane_kernel=kind) as nl:
        assert (nl.query(7), nl.query(8)) == ((1.0, float(kind)) if kind != 3 else (0.0, 0.0))   # the requested kernel runs
    with GeneNL(wl) as nl:
        assert nl.query(8) == 2.0                                   # and the group kernel is the default at this size
    check_parity(wl, cuda_device, plane_kernel=kind)
    check_parity(wl, cuda_device, plane_kernel=kind, scratch_bytes=20 << 20)   # several launches
    check_parity(wl, cuda_device, plane_kernel=kind, host=True)                 # behind the streaming driver


@pytest.mark.parametrize("kind", SPREAD_KINDS)
def test_spread_kernels_config2_full_size_all_planes(cuda_device, kind):
    _full_size(cuda_device, 2, None, plane_kernel=kind)


# 768 x 384 planes (the shape of configs[3]): group kernel (2, the default), batched kernels (3: k_xinv<768,...,SEQ> +
# k_ybracket<384> + k_xfwd<768>), warp-autonomous form (4).  40 planes > 2 x 18 groups of 8 CTAs, and the real-space chi
# rows of the chunk (10 planes x 4.7 MB) exceed 40 MB, so that k_ybracket<384> takes its v-fastest tile walk under kind 3.
@pytest.mark.parametrize("kind", [2, 3, 4])
@pytest.mark.parametrize("nz,nv,nw,nspec", [(1, 1, 1, 1), (10, 4, 1, 1), (2, 3, 2, 2)])
def test_768x384_kernel_families(cuda_device, nz, nv, nw, nspec, kind):
    from paper_1310_1485_b200 import GeneNL
    wl = W.small_workload(512, 128, nz, nv, nw, nspec, 0.0125, 0.025, False, seed=700 + nz + nv)
    with GeneNL(wl, plane_kernel=kind) as nl:
        assert (nl.query(7), nl.query(8)) == ((1.0, float(kind)) if kind != 3 else (0.0, 0.0))
    with GeneNL(wl) as nl:
        assert nl.query(8) == 2.0
    check_parity(wl, cuda_device, plane_kernel=kind)
    if nz * nv > 1:
        check_parity(wl, cuda_device, plane_kernel=kind, scratch_bytes=40 << 20)   # several launches / ragged batches


@pytest.mark.parametrize("kind", [3, 4])
def test_config3_full_size_sampled_planes_other_kernel_families(cuda_device, kind):
    """The full-size runs BASELINE.md quotes for the batched and the warp-autonomous kernels at configs[3]."""
    _full_size(cuda_device, 3, 96, plane_kernel=kind)


def test_config4_full_size_sampled_planes_warp_kernel(cuda_device):
    _full_size(cuda_device, 4, 160, plane_kernel=4)


@pytest.mark.parametrize("kind", SPREAD_KINDS)
def test_spread_kernels_properties_and_selection(cuda_device, kind):
    from paper_1310_1485_b200 import (GENE_NL_KERNEL_AUTO, GENE_NL_KERNEL_BATCHED, GENE_NL_KERNEL_CLUSTER, GeneNL,
                                      GeneNLError, gene_nl_set_plane_kernel)
    GENE_NL_KERNEL_CLUSTER = kind   # noqa: N806  (the body below is written for "the selected kind")
    wl = W.small_workload(256, 64, 2, 3, 1, 2, 0.05, 0.05, False, seed=61)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    kw = dict(plane_kernel=GENE_NL_KERNEL_CLUSTER)
    assert torch.equal(gpu_compute(wl, chi, g, rhs, scale=0.0, **kw), rhs)          # scale = 0: bit-identical
    a = gpu_compute(wl, chi, g, rhs, **kw)
    assert torch.equal(a, gpu_compute(wl, chi, g, rhs, **kw))                       # deterministic
    b = gpu_compute(wl, chi, g, rhs, plane_kernel=GENE_NL_KERNEL_BATCHED)           # the batched kernels
    assert (a - b).abs().max() <= 1e-13 * (b - rhs).abs().max()
    h = wl.nx0 // 2
    assert torch.equal(W.as_planes(a, wl)[:, :, h], W.as_planes(rhs, wl)[:, :, h])  # Nyquist row untouched
    with GeneNL(wl) as nl:                                                          # switching back and forth on one plan
        gene_nl_set_plane_kernel(nl.h, GENE_NL_KERNEL_CLUSTER)
        out = rhs.clone()
        nl.compute(chi, g, out)
        torch.cuda.synchronize()
        assert torch.equal(out, a)
        gene_nl_set_plane_kernel(nl.h, GENE_NL_KERNEL_BATCHED)
        assert nl.query(7) == 0.0 and nl.query(8) == 0.0
        out = rhs.clone()
        nl.compute(chi, g, out)
        torch.cuda.synchronize()
        assert torch.equal(out, b)
        gene_nl_set_plane_kernel(nl.h, GENE_NL_KERNEL_AUTO)
        out = rhs.clone()
        nl.compute(chi, g, out)
        torch.cuda.synchronize()
        assert (out - b).abs().max() <= 1e-13 * (b - rhs).abs().max()
        with pytest.raises(GeneNLError):
            gene_nl_set_plane_kernel(nl.h, 7)
    for bad in (W.small_workload(128, 32, 1, 1, 1, 1), W.small_workload(256, 64, 1, 1, 1, 1, chi_has_v=True)):
        with GeneNL(bad) as nl:
            if kind == GENE_NL_KERNEL_BATCHED:
                gene_nl_set_plane_kernel(nl.h, kind)                                    # the batched kernels serve every size
            else:
                with pytest.raises(GeneNLError):
                    gene_nl_set_plane_kernel(nl.h, GENE_NL_KERNEL_CLUSTER)              # no cluster / group kernel for these


# 144 x 144 planes (the shape of configs[4]): the group kernel with chi per plane (chi goes through the kernel like g) and
# with chi shared over v, and the batched kernels on the same data
@pytest.mark.parametrize("kind", [2, 3, 4])
@pytest.mark.parametrize("chi_has_v", [True, False])
@pytest.mark.parametrize("nz,nv,nw,nspec", [(1, 1, 1, 1), (3, 5, 2, 2), (37, 2, 1, 1),
                                            (37, 9, 1, 1)])   # 333 planes > 2 x 148 groups: second and third plane per group
def test_group_kernel_144x144_planes(cuda_device, nz, nv, nw, nspec, chi_has_v, kind):
    from paper_1310_1485_b200 import GeneNL
    wl = W.small_workload(96, 48, nz, nv, nw, nspec, 0.04, 0.06, chi_has_v, seed=400 + nz + nv)
    with GeneNL(wl) as nl:
        assert nl.query(8) == 2.0                                   # the group kernel is the default at this size
    check_parity(wl, cuda_device, plane_kernel=kind)
    check_parity(wl, cuda_device, plane_kernel=kind, scratch_bytes=4 << 20)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    a = gpu_compute(wl, chi, g, rhs, plane_kernel=2)
    b = gpu_compute(wl, chi, g, rhs, plane_kernel=3)
    assert (a - b).abs().max() <= 1e-13 * (b - rhs).abs().max()
    assert torch.equal(gpu_compute(wl, chi, g, rhs, scale=0.0, plane_kernel=kind), rhs)


# nw is chosen so that 3 * 5 * nw planes give every persistent CTA / cluster / group at least three planes (148 CTAs or
# groups of one CTA: 450 planes; 37 groups of four: 120; 18 groups of eight and 15 clusters of eight: 60): the plane loop's
# phase flips, the request of the next plane's first block and the dropped scratch lines are all exercised under
# co-scheduling, not only a group's first plane
@pytest.mark.parametrize("nx0,nky0,chi_has_v,kind,nw", [
    (128, 32, False, None, 30),  # k_plane_fused2: __syncwarp-only chains over in-place tiles, shadow lanes
    (16, 8, False, None, 30),    # k_plane_fused (first generation)
    (256, 64, False, 2, 8),      # k_plane_group: hand-overs through L2, counters, bulk copies into live tiles
    (256, 64, False, 1, 4),      # k_plane_cluster: DSMEM stores + mbarrier transaction counts
    (96, 48, True, 2, 30),       # k_plane_group with chi per plane (groups of one CTA)
    (96, 48, False, 2, 30),      # k_plane_group with chi shared over v (groups of one CTA)
    (512, 128, False, 2, 4),     # k_plane_group, radix-16 second y stage
    (256, 64, True, 3, 2),       # batched kernels
    (256, 64, False, 4, 8),      # k_plane_wa: per-warp tiles, every warp on the hand-over counters
    (96, 48, True, 4, 30),       # k_plane_wa with chi per plane
    (512, 128, False, 4, 4),     # k_plane_wa, radix-32 x stages
])
def test_repeated_runs_give_the_same_bits(cuda_device, nx0, nky0, chi_has_v, kind, nw):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.md), so a data race in the shared-memory /
    distributed-shared-memory / L2 hand-overs has to show up here: the kernels are deterministic by construction (no
    atomics on data, fixed summation order), so 24 runs under different co-scheduling -- alone, behind a memory-bound
    kernel on another stream, with a different number of planes in flight -- must agree with the first one bit for bit,
    and that one with the oracle."""
    from paper_1310_1485_b200 import GeneNL
    wl = W.small_workload(nx0, nky0, 3, 5, nw, 1, 0.04, 0.05, chi_has_v, seed=500 + nx0)
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    check_parity(wl, cuda_device, plane_kernel=kind)
    junk = torch.empty(64 << 20, dtype=torch.float64, device=cuda_device)
    side = torch.cuda.Stream()
    with GeneNL(wl, plane_kernel=kind) as nl:
        first = rhs.clone()
        nl.compute(chi, g, first)
        torch.cuda.synchronize()
        for rep in range(24):
            out = rhs.clone()
            if rep % 3 == 1:
                with torch.cuda.stream(side):
                    junk.mul_(1.0000001)                 # a bandwidth hog next to the kernels
            nl.compute(chi, g, out)
            torch.cuda.synchronize()
            assert torch.equal(out, first), f"run {rep} differs"
    half = W.small_workload(nx0, nky0, 3, 5, nw // 2, 1, 0.04, 0.05, chi_has_v, seed=500 + nx0)   # first half of the (w,s) slabs
    sub, cs, gs, rs = W.shard_arrays(wl, chi, g, rhs, 0, 2)
    assert sub.planes == half.planes
    part = gpu_compute(sub, cs.contiguous(), gs.contiguous(), rs.contiguous(), plane_kernel=kind)
    assert torch.equal(part.reshape(-1), first.reshape(2, -1)[0])


def test_config1_sampled_modes_against_the_definition(cuda_device):
    """Sampled outputs the definition can compute one by one, at BASELINE.json's full size."""
    wl = W.CONFIGS[1]
    chi, g, rhs = W.make_inputs(wl, cuda_device)
    out = gpu_compute(wl, chi, g, rhs)
    ii = np.array([0, 1, 63, 65, 127, 17, 100, 40, 5, 90])
    jj = np.array([0, 31, 5, 0, 31, 16, 1, 30, 0, 12])
    for p in sample_planes(wl, 6, seed=1):
        X = W.as_planes(chi, wl)[W.chi_plane_of(wl, int(p))].cpu().numpy()
        G = W.as_planes(g, wl)[int(p)].cpu().numpy()
        N = oracle.nl_convolution_modes(X, G, wl.kxmin, wl.kymin, ii, jj)
        d = (W.as_planes(out, wl)[int(p)] - W.as_planes(rhs, wl)[int(p)]).cpu().numpy()[jj, ii]
        assert np.abs(d - wl.scale * N).max() <= 1e-11 * np.abs(N).max()


def test_compute_is_capturable_in_a_cuda_graph(cuda_device):
    """gene_nl_compute only enqueues kernels on the caller's stream (no synchronisation, no allocation): it can be
    captured into a CUDA graph and replayed; fused and batched paths."""
    from paper_1310_1485_b200 import GeneNL
    from paper_1310_1485_b200 import GENE_NL_KERNEL_CLUSTER, GENE_NL_KERNEL_GROUP
    for wl, pk in ((W.small_workload(128, 32, 2, 3, 1, 1, 0.05, 0.05, False, seed=41), None),     # fused kernel
                   (W.small_workload(256, 64, 2, 2, 1, 2, 0.05, 0.05, True, seed=42), None),      # batched kernels
                   (W.small_workload(256, 64, 2, 2, 1, 2, 0.05, 0.05, False, seed=43), GENE_NL_KERNEL_CLUSTER),
                   (W.small_workload(256, 64, 2, 2, 1, 2, 0.05, 0.05, False, seed=44), GENE_NL_KERNEL_GROUP)):
        chi, g, rhs = W.make_inputs(wl, cuda_device)
        expect = gpu_compute(wl, chi, g, rhs, plane_kernel=pk)
        out = rhs.clone()
        with GeneNL(wl, plane_kernel=pk) as nl:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                nl.compute(chi, g, out.clone())          # warm-up outside capture
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                nl.compute(chi, g, out)                   # torch's capture stream is the current stream here
            assert torch.equal(out, rhs)                  # nothing ran during capture
            graph.replay()
            torch.cuda.synchronize()
            assert torch.equal(out, expect)
            graph.replay()                                # rhs keeps accumulating: out = rhs + 2 scale N
            torch.cuda.synchronize()
            d = (out - rhs) - 2 * (expect - rhs)
            assert d.abs().max() <= 1e-13 * (expect - rhs).abs().max()
