"""Multi-rank host logic on CPU (gloo, world_size 2): the plane sharding of SURVEY.md 8(e) covers every
(w,s) slab exactly once with chi sharded alongside g, the sharded oracle results assemble to the
unsharded one (no exchange on the data path), and the bench's timing reduction is a max over ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1310_1485_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.small_workload(16, 8, 2, 3, 3, 1, 0.1, 0.1, False, seed=31)   # 3 slabs over 2 ranks: ragged
        chi, g, rhs = W.make_inputs(wl)                                   # same seed on every rank
        sub, cs, gs, rs = W.shard_arrays(wl, chi, g, rhs, rank, world)
        ci = np.array([W.chi_plane_of(sub, p) for p in range(sub.planes)])
        out = oracle.nl_pseudospectral(W.as_planes(cs, sub).numpy(), W.as_planes(gs, sub).numpy(),
                                       W.as_planes(rs, sub).numpy(), wl.scale, wl.kxmin, wl.kymin, ci)
        # gather the shards (test harness only -- the data path itself has no collective)
        s0, s1 = W.shard_slabs(wl, rank, world)
        full = torch.zeros((wl.planes, wl.nky0, wl.nx0), dtype=torch.complex128)
        per_slab = wl.nz * wl.nv
        full[s0 * per_slab:s1 * per_slab] = torch.from_numpy(out)
        buf = torch.view_as_real(full).contiguous()
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
        ms = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)      # per-rank step time
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        if rank == 0:
            cif = np.array([W.chi_plane_of(wl, p) for p in range(wl.planes)])
            ref = oracle.nl_pseudospectral(W.as_planes(chi, wl).numpy(), W.as_planes(g, wl).numpy(),
                                           W.as_planes(rhs, wl).numpy(), wl.scale, wl.kxmin, wl.kymin, cif)
            got = torch.view_as_complex(buf).numpy()
            ret["equal"] = bool(np.array_equal(got, ref))
            ret["ms"] = float(ms.item())
    finally:
        dist.destroy_process_group()


def test_sharded_planes_assemble_to_the_unsharded_result_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
        assert ret["equal"] is True
        assert ret["ms"] == 15.0


def test_shard_slabs_partition():
    for nw, nspec, world in [(8, 2, 1), (8, 2, 2), (8, 2, 4), (8, 2, 8), (3, 1, 2), (16, 3, 8), (1, 1, 4)]:
        wl = W.small_workload(16, 8, 2, 2, nw, nspec)
        seen = []
        for r in range(world):
            s0, s1 = W.shard_slabs(wl, r, world)
            assert 0 <= s0 <= s1 <= nw * nspec
            seen += list(range(s0, s1))
        assert seen == list(range(nw * nspec))
