#!/usr/bin/env python
"""bench.py -- E x B nonlinearity planes/s on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py --gpus N --steps K --warmup W [--config I] [--impl reference]

A "step" is one pass of the whole hot path (gene_nl_compute: derivative + pad + to real space,
bracket, back, delete modes, prefactor, add to rhs) over all planes of the workload.  The workload is
BASELINE.json configs[3] (512x128 modes, 24 576 planes, 24 GiB per array): BASELINE.json's metric names
no configuration, so the headline is the largest single-GPU one; with no --config the line also carries
`per_config` = configs[1], [2], [4] measured device-resident in the same run.  For N > 1 (torchrun, one
rank per GPU) every rank runs its own problem of that size (planes are independent: weak scaling, no
collective on the data path); the time is the max over ranks.

Keys beyond the base contract: `roofline` (dominant kernel, timed live with CUDA events on the
launching stream through gene_nl_compute_profiled), `roofline_step` (whole step), `kernels`
(per-class device time), `cpu_baseline` (the oracle on the host cores, bounded sample), `e2e`
(gene_nl_compute_host on pinned host buffers, copies inside the timed region), `clocks`.
`--impl reference` times the CPU oracle as it stands (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ExB nonlinearity planes/s"
UNIT = "planes/s"
# FP64 ALU peak model: 148 SMs x 64 FP64 FMA lanes/SM/clk x 2 flop x 1.965 GHz (DESIGN.md sect. 7)
FP64_LANES_PER_SM = 64


def per_kernel_flops(wl, fused=False):
    """Conventional flop split of SURVEY.md 8(d)'s F over the four kernel classes (DESIGN.md sect. 7)."""
    Nx, Ny, M = wl.Nx, wl.Ny, wl.nx0 * wl.nky0
    x1 = wl.nky0 * 5.0 * Nx * math.log2(Nx)      # x half of one 2-D transform (nky0 live columns)
    y1 = Nx * 2.5 * Ny * math.log2(Ny)           # y half of one real 2-D transform
    P, Q = wl.planes, wl.chi_planes
    per_plane = {
        "k_xinv": 2 * x1 + 4 * M,                # derivative (2 mult/value) + two x-syntheses
        "k_yreal": 2 * y1,                       # two real y-syntheses (dx chi, dy chi)
        "k_ybracket": 3 * y1 + 3 * Nx * Ny,      # two y-syntheses, bracket, one y-analysis
        "k_xfwd": x1 + 4 * M,                    # x-analysis + scale/accumulate (2 FMA/value)
    }
    if fused:  # the g side of a plane runs in one kernel; k_xinv / k_yreal only see chi
        return {"k_xinv": Q * per_plane["k_xinv"], "k_yreal": Q * per_plane["k_yreal"],
                "k_plane_fused": P * (per_plane["k_xinv"] + per_plane["k_ybracket"] + per_plane["k_xfwd"])}
    return {"k_xinv": (P + Q) * per_plane["k_xinv"], "k_yreal": Q * per_plane["k_yreal"],
            "k_ybracket": P * per_plane["k_ybracket"], "k_xfwd": P * per_plane["k_xfwd"]}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, torch_index, period=0.002):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.max_mhz = period, [], set(), None
        self._halt = threading.Event()
        self.h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            uuid = str(torch.cuda.get_device_properties(torch_index).uuid)
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid).encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(torch_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def run(self):
        if self.h is None:
            return
        while not self._halt.is_set():
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                bits = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            self._halt.wait(self.period)

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def time_oracle(wl, seconds, threads):
    """The oracle as it stands on a bounded sample of the workload (`seconds` of wall time on `threads`
    cores): returns (planes/s, planes, elapsed)."""
    import numpy as np
    import torch

    import oracle
    from paper_1310_1485_b200 import workloads as W

    # inputs for slabs that contain the sampled planes: up to four (w,s) slabs of the workload's shape
    sub = W.Workload(wl.name + "_slab", wl.nx0, wl.nky0, wl.nz, wl.nv, min(wl.nw, 4), 1, wl.kxmin, wl.kymin,
                     wl.chi_has_v, wl.seed, wl.rhs_random, wl.scale)
    chi, g, rhs = W.make_inputs(sub, "cpu")
    G, X, R = (W.as_planes(t, sub).numpy() for t in (g, chi, rhs))
    ci = np.array([W.chi_plane_of(sub, p) for p in range(sub.planes)])

    def run(n):
        n = min(n, sub.planes)
        t0 = time.perf_counter()
        oracle.nl_pseudospectral(X, G[:n], R[:n], wl.scale, wl.kxmin, wl.kymin, ci[:n])
        return n, time.perf_counter() - t0

    run(threads)                                # warm-up (thread pool, page faults)
    n, dt = run(4 * threads)                    # calibration: four planes per thread
    want = int(max(threads, min(sub.planes, n / dt * seconds)))
    want -= want % threads
    n, dt = run(max(want, threads))
    return n / dt, n, dt


def reference_arm(args, wl):
    """`--impl reference`: the CPU oracle, as it stands, on the host cores; rank 0 only."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np

    from paper_1310_1485_b200 import workloads as W
    threads = oracle.num_threads()
    sub = W.Workload(wl.name + "_slab", wl.nx0, wl.nky0, wl.nz, wl.nv, 1, 1, wl.kxmin, wl.kymin,
                     wl.chi_has_v, wl.seed, wl.rhs_random, wl.scale)
    chi, g, rhs = W.make_inputs(sub, "cpu")
    G, X, R = (W.as_planes(t, sub).numpy() for t in (g, chi, rhs))
    ci = np.array([W.chi_plane_of(sub, p) for p in range(sub.planes)])
    t0 = time.perf_counter()
    oracle.nl_pseudospectral(X, G[:threads], R[:threads], wl.scale, wl.kxmin, wl.kymin, ci[:threads])
    rate = threads / (time.perf_counter() - t0)
    total_steps = args.steps + args.warmup
    n = int(min(sub.planes, max(threads, rate * 100.0 / max(total_steps, 1))))
    n -= n % threads
    n = max(n, threads)
    for _ in range(args.warmup):
        oracle.nl_pseudospectral(X, G[:n], R[:n], wl.scale, wl.kxmin, wl.kymin, ci[:n])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.nl_pseudospectral(X, G[:n], R[:n], wl.scale, wl.kxmin, wl.kymin, ci[:n])
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = f"{n} planes of {wl.name} per step (one (w,s) slab), recursive radix-2/3 FFT oracle"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "planes_per_step": n, "nx0": wl.nx0, "nky0": wl.nky0},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def xglobal_main(args):
    """`--xglobal`: the x-global variant, the operator and plane shape the paper timed
    (64 x 16 planes, 589 824 of them device-resident: Table 4).  HBM bound: 6 planes of traffic per
    plane, so the roofline is bytes / measured HBM bandwidth."""
    import numpy as np
    import torch

    from paper_1310_1485_b200 import gene_nlx_compute, gene_nlx_create, gene_nlx_destroy, gene_nlx_query
    from paper_1310_1485_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    base = W.XGLOBAL_PAPER
    wl = W.XGlobalWorkload(base.name if args.xglobal_planes == base.planes else f"xglobal_64x16_{args.xglobal_planes}",
                           base.nx, base.nky0, args.xglobal_planes, base.seed + 1000 * rank, base.scale)
    if args.impl == "reference":
        if rank != 0:
            return
        import oracle
        threads = oracle.num_threads()
        n = 16384
        sub = W.XGlobalWorkload("sample", wl.nx, wl.nky0, n, wl.seed, wl.scale)
        a, b, c, d, pref, r = (t.numpy() for t in W.make_xglobal_inputs(sub, "cpu"))
        for _ in range(args.warmup):
            oracle.nlx_pseudospectral(a, b, c, d, pref, r, wl.scale)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            oracle.nlx_pseudospectral(a, b, c, d, pref, r, wl.scale)
        dt = time.perf_counter() - t0
        value = n * args.steps / dt
        sample = f"{n} planes of 64x16 per step, recursive radix-2/3 FFT oracle"
        print(json.dumps({
            "impl": "reference", "metric": "x-global ExB nonlinearity planes/s (P_c/s)", "value": value, "unit": UNIT,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": value / 197e3, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wl.name, "planes_per_step": n, "nx": wl.nx, "nky0": wl.nky0},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}), flush=True)
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    vex, vey, dxg, dyg, pref, rhs = W.make_xglobal_inputs(wl, dev)
    h = gene_nlx_create(wl.nx, wl.nky0, wl.planes)
    stream = torch.cuda.current_stream()
    for _ in range(max(args.warmup, 3)):
        gene_nlx_compute(h, vex, vey, dxg, dyg, pref, rhs, wl.scale, stream)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        gene_nlx_compute(h, vex, vey, dxg, dyg, pref, rhs, wl.scale, stream)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item()) / args.steps
    value = wl.planes * world / (ms_per_step * 1e-3)
    B, F = gene_nlx_query(h, 5), gene_nlx_query(h, 6)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    gbs = B * wl.planes / (ms_per_step * 1e-3) / 1e9     # the step IS one launch of k_xglobal
    cap, why = measured_traffic("xglobal_64x16")
    traffic = cap["k_xglobal"][0] * wl.planes / cap["k_xglobal"][1] if "k_xglobal" in cap else None
    roofline = {"kernel": "k_xglobal", "bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                "frac": gbs / hbm_peak, "traffic": traffic,
                "traffic_note": why or ("ncu dram__bytes capture of one whole step (profiles/r03_dram.md), stamped with src_sha16 %s" % source_sha16()),
                "peak_source": "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s",
                "bytes_per_plane": B, "flops_per_plane": F, "achieved_tflops": F * wl.planes / (ms_per_step * 1e-3) / 1e12,
                "share_of_step": 1.0}
    # end to end: pinned host buffers, H2D of the five arrays and D2H of rhs inside the timed region (bounded slice)
    e2e = None
    if not args.no_e2e:
        from paper_1310_1485_b200 import gene_nlx_compute_host
        n = min(wl.planes, 65536)
        host = [t[:n].cpu().pin_memory() for t in (vex, vey, dxg, dyg, rhs)]
        hpref = pref.cpu()
        h2 = gene_nlx_create(wl.nx, wl.nky0, n)

        def once():   # chunks of planes on three streams: H2D, kernel and D2H of different chunks overlap
            gene_nlx_compute_host(h2, host[0], host[1], host[2], host[3], hpref, host[4], wl.scale)
        once()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            once()
        barrier()
        dt = time.perf_counter() - t0
        # the paper's own roofline for this path, redrawn: what the host link alone allows.  Measured
        # here with plain pinned copies of one array (CUDA events), not taken from a data sheet.
        def link_gbs(dst, src):
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            dst.copy_(src, non_blocking=True)
            torch.cuda.synchronize()
            ev0.record()
            for _ in range(3):
                dst.copy_(src, non_blocking=True)
            ev1.record()
            torch.cuda.synchronize()
            return 3 * src.numel() * src.element_size() / (ev0.elapsed_time(ev1) * 1e-3) / 1e9
        dev_buf = torch.empty_like(host[0], device=dev)
        h2d, d2h = link_gbs(dev_buf, host[0]), link_gbs(host[0].clone().pin_memory(), dev_buf)
        del dev_buf
        U = wl.plane_bytes
        e2e = {"value": n * world * args.e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": 5 * n * wl.plane_bytes,
               "d2h_bytes_per_step": n * wl.plane_bytes, "steps": args.e2e_steps,
               "api": f"gene_nlx_compute_host on {n} planes (pinned host buffers, chunked over three streams)",
               "link_h2d_gbs": h2d, "link_d2h_gbs": d2h,
               # full duplex: 5 planes in and 1 plane out per plane computed move at the same time
               "link_roofline_planes_per_s": world / max(5 * U / (h2d * 1e9), U / (d2h * 1e9)),
               # the paper's model: BW0 / 6 (transferable planes per second times the intensity 1/6, half duplex)
               "paper_model_planes_per_s": world * h2d * 1e9 / (6 * U)}
        gene_nlx_destroy(h2)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        n = 32768
        sub = W.XGlobalWorkload("sample", wl.nx, wl.nky0, n, wl.seed, wl.scale)
        a, b, c, d, pr, r = (t.numpy() for t in W.make_xglobal_inputs(sub, "cpu"))
        t0 = time.perf_counter()
        oracle.nlx_pseudospectral(a, b, c, d, pr, r, wl.scale)
        dt = time.perf_counter() - t0
        cpu = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{n} planes of 64x16, {dt:.1f} s wall"}
    gene_nlx_destroy(h)
    if rank == 0:
        print(json.dumps({
            "metric": "x-global ExB nonlinearity planes/s (P_c/s)", "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": value / 197e3, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "nx": wl.nx, "nky0": wl.nky0, "planes_per_gpu": wl.planes,
                       "padded_y": wl.Ny, "cache": f"inputs larger than L2 ({6 * wl.planes * wl.plane_bytes / 2**30:.1f} GiB per GPU)",
                       "baseline": "PAPER.md:98-105 Table 4: 197 kP_c/s on one K20X, device-resident (another machine: context)",
                       "parallelism": f"planes x{world} (independent problems per GPU)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps, "roofline": roofline, "cpu_baseline": cpu}), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def em_main(args):
    """`--em`: configs[args.config]'s grid with chi composed on the device from phi_bar and A_par_bar
    (gene_nl_compute_em).  Same metric; the per-plane chi array is never formed."""
    import numpy as np
    import torch

    from paper_1310_1485_b200 import (GENE_NL_CHI_EM, gene_nl_compute_em, gene_nl_create, gene_nl_destroy,
                                      gene_nl_launches_per_compute, gene_nl_query)
    from paper_1310_1485_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    c = W.CONFIGS[args.config]
    wl = W.Workload(c.name + "_em_composed", c.nx0, c.nky0, c.nz, c.nv, c.nw, c.nspec, c.kxmin, c.kymin, False,
                    c.seed + 1000 * rank, c.rhs_random, c.scale)
    wl2 = W.Workload(wl.name + "_apar", c.nx0, c.nky0, c.nz, c.nv, c.nw, c.nspec, c.kxmin, c.kymin, False,
                     c.seed + 77 + 1000 * rank, c.rhs_random, c.scale)
    vpar = np.concatenate([np.linspace(-3.0, 3.0, c.nv) * (1.0 + 0.5 * s) for s in range(c.nspec)])
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    phi, g, rhs = W.make_inputs(wl, dev)
    apar, _, _ = W.make_inputs(wl2, dev)
    del _
    h = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, GENE_NL_CHI_EM)
    stream = torch.cuda.current_stream()
    for _ in range(max(args.warmup, 3)):
        gene_nl_compute_em(h, phi, apar, vpar, g, rhs, wl.scale, stream)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        gene_nl_compute_em(h, phi, apar, vpar, g, rhs, wl.scale, stream)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item()) / args.steps
    value = wl.planes * world / (ms_per_step * 1e-3)
    F, B = gene_nl_query(h, 6), gene_nl_query(h, 5)
    fp64_model = 148 * FP64_LANES_PER_SM * 2 * 1.965e9 / 1e12
    tf = F * wl.planes / (ms_per_step * 1e-3) / 1e12
    kind = {0.0: "batched kernels (k_xinv, k_ybracket<EM>, k_xfwd)", 2.0: "group kernel k_plane_group<EM>"}.get(gene_nl_query(h, 8), "?")
    roofline = {"kernel": f"whole step: {kind}; chi side: k_xinv + k_yreal on phi_bar and A_par_bar", "bound": "alu",
                "achieved": tf, "peak": fp64_model, "unit": "TFLOP/s", "frac": tf / fp64_model, "traffic": None,
                "peak_source": "model 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md sect. 7)",
                "flops_per_plane": F, "bytes_per_plane": B}
    e2e = None
    if not args.no_e2e:   # pinned host buffers; H2D of g, rhs, phi, apar and D2H of rhs inside the timed region
        from paper_1310_1485_b200 import gene_nl_compute_em_host
        host = [t.cpu().pin_memory() for t in (phi, apar, g, rhs)]

        def once():
            gene_nl_compute_em_host(h, host[0], host[1], vpar, host[2], host[3], wl.scale)
        once()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            once()
        barrier()
        dt = time.perf_counter() - t0
        nb = sum(t.numel() * 16 for t in (phi, apar, g, rhs))
        e2e = {"value": wl.planes * world * args.e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": nb,
               "d2h_bytes_per_step": rhs.numel() * 16, "steps": args.e2e_steps,
               "api": "gene_nl_compute_em_host (pinned host buffers, one (w,s) slab per stage, three streams)"}
    launches = gene_nl_launches_per_compute(h)
    gene_nl_destroy(h)
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "nx0": wl.nx0, "nky0": wl.nky0, "planes_per_gpu": wl.planes,
                       "chi": "composed on device: phi_bar - v_par * A_par_bar (gene_nl_compute_em)",
                       "cache": "inputs larger than L2", "parallelism": f"planes x{world} (independent problems per GPU)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches * args.steps, "roofline": roofline,
            "cpu_baseline": None}), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def plane_kernel_name(wl, fused, kind, em=False):
    """The instantiation gene_nl_create / gene_nl_set_plane_kernel selected for this plane shape (the tables find_fused2,
    find_fused, find_group, find_wa, find_cluster of csrc/gene_nl.cu), from gene_nl_query(h, 7) and (h, 8): the roofline
    line names the kernel that ran, not its class."""
    nx, ny = wl.Nx, wl.Ny
    chiv = bool(wl.chi_has_v) and not em
    tail = ",EM" if em else (",CHIV" if chiv else "")
    if not fused:
        return None
    if kind == 2.0:
        return {(384, 192): "k_plane_group<24,16,24,G=4,NH=2%s>", (768, 384): "k_plane_group<48,16,24,G=8,NH=4,BY=16,X2=24x32%s>",
                (144, 144): "k_plane_group<12,12,18,G=1%s>"}.get((nx, ny), "k_plane_group<?%s>") % tail
    if kind == 4.0:
        return {(384, 192): "k_plane_wa<24,16,24,8,G=4%s>", (768, 384): "k_plane_wa<24,32,24,16,G=8%s>",
                (144, 144): "k_plane_wa<12,12,18,8,G=1%s>"}.get((nx, ny), "k_plane_wa<?%s>") % tail
    if kind == 1.0:
        return "k_plane_cluster<24,16,24,C=8>"
    if ny == 96 and nx in (48, 96, 192):
        return "k_plane_fused2<%d,12,8>" % (nx // 8)
    return "k_plane_fused<%d,%d,8>" % (nx // 8, ny // 8)


def side_xglobal(dev, peaks, planes=65536, steps=10):
    """Device-resident x-global step on a slice of the paper's workload, for the compact summary of the
    default run; `bench.py --xglobal` is the full measurement (589 824 planes, e2e, cpu_baseline)."""
    import torch
    from paper_1310_1485_b200 import gene_nlx_compute, gene_nlx_create, gene_nlx_destroy, gene_nlx_query
    from paper_1310_1485_b200 import workloads as W
    base = W.XGLOBAL_PAPER
    wl = W.XGlobalWorkload(f"xglobal_64x16_{planes}", base.nx, base.nky0, planes, base.seed, base.scale)
    arrs = W.make_xglobal_inputs(wl, dev)
    h = gene_nlx_create(wl.nx, wl.nky0, wl.planes)
    stream = torch.cuda.current_stream()
    for _ in range(3):
        gene_nlx_compute(h, *arrs, wl.scale, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        gene_nlx_compute(h, *arrs, wl.scale, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    gbs = gene_nlx_query(h, 5) * wl.planes / (ms * 1e-3) / 1e9
    gene_nlx_destroy(h)
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    return {"kernel": "k_xglobal<48,6,8,64,16>", "bound": "hbm", "frac": gbs / hbm_peak, "achieved_gbs": gbs, "peak_gbs": hbm_peak,
            "ms": ms, "planes": planes, "planes_per_s": planes / (ms * 1e-3), "gpu_launches": steps}


def side_em(dev, idx=4, steps=5):
    """Device-resident EM step (chi composed on the device) on configs[idx]'s grid, for the compact summary
    of the default run; `bench.py --em` is the full measurement."""
    import numpy as np
    import torch
    from paper_1310_1485_b200 import (GENE_NL_CHI_EM, gene_nl_compute_em, gene_nl_create, gene_nl_destroy,
                                      gene_nl_launches_per_compute, gene_nl_query)
    from paper_1310_1485_b200 import workloads as W
    c = W.CONFIGS[idx]
    wl = W.Workload(c.name + "_em_composed", c.nx0, c.nky0, c.nz, c.nv, c.nw, c.nspec, c.kxmin, c.kymin, False, c.seed,
                    c.rhs_random, c.scale)
    wl2 = W.Workload(wl.name + "_apar", c.nx0, c.nky0, c.nz, c.nv, c.nw, c.nspec, c.kxmin, c.kymin, False, c.seed + 77,
                     c.rhs_random, c.scale)
    vpar = np.concatenate([np.linspace(-3.0, 3.0, c.nv) * (1.0 + 0.5 * s) for s in range(c.nspec)])
    phi, g, rhs = W.make_inputs(wl, dev)
    apar = W.make_inputs(wl2, dev)[0]
    h = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, GENE_NL_CHI_EM)
    stream = torch.cuda.current_stream()
    for _ in range(3):
        gene_nl_compute_em(h, phi, apar, vpar, g, rhs, wl.scale, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        gene_nl_compute_em(h, phi, apar, vpar, g, rhs, wl.scale, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    fp64_model = 148 * FP64_LANES_PER_SM * 2 * 1.965e9 / 1e12
    tf = gene_nl_query(h, 6) * wl.planes / (ms * 1e-3) / 1e12
    name = plane_kernel_name(wl, gene_nl_query(h, 7) == 1.0, gene_nl_query(h, 8), em=True) or "k_xinv + k_ybracket<EM> + k_xfwd"
    launches = gene_nl_launches_per_compute(h) * steps
    gene_nl_destroy(h)
    return {"kernel": name, "bound": "alu", "step_frac": tf / fp64_model, "achieved_tflops": tf, "ms": ms, "planes": wl.planes,
            "planes_per_s": wl.planes / (ms * 1e-3), "gpu_launches": launches,
            "note": "whole step incl. the chi-side launches on phi_bar and A_par_bar"}


def source_sha16():
    """sha256 over the CUDA sources: rows of profiles/dram_traffic.csv are stamped with it at capture time."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1310_1485_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def measured_traffic(workload_name):
    """{kernel: (dram bytes per launch, planes per launch)} from the committed ncu capture, ONLY when the capture was
    taken from the CUDA sources that are being timed now (src_sha16 column); else ({}, why)."""
    import csv
    rows, stale = {}, 0
    try:
        sha = source_sha16()
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "dram_traffic.csv"))):
            if row["workload"] != workload_name:
                continue
            if row.get("src_sha16", "") != sha:
                stale += 1
                continue
            rows[row["kernel"]] = (float(row["dram_bytes_per_launch"]), float(row["planes_per_launch"]))
    except Exception as e:  # noqa: BLE001
        return {}, f"profiles/dram_traffic.csv unreadable: {e}"
    if not rows:
        return {}, ("capture predates the current CUDA sources" if stale else "no ncu capture for this workload")
    return rows, None


def run_config(wl, args, env, do_e2e, do_cpu, headline, plane_kernel=None):
    """Time one workload: device-resident steps (CUDA events on the launching stream, max over ranks), per-kernel
    rooflines (event pair per launch), e2e through the host entry point, the oracle as cpu_baseline."""
    import torch

    from paper_1310_1485_b200 import GeneNL, gene_nl_probe_peaks
    from paper_1310_1485_b200 import workloads as W
    from paper_1310_1485_b200.binding import KERNEL_CLASSES

    dev, dist, world, rank, local_rank = env["dev"], env["dist"], env["world"], env["rank"], env["local_rank"]

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    strong = args.strong and world > 1
    if strong:
        # ONE problem of the workload's shape, its (w,s) slabs sharded over the ranks: g, rhs and
        # chi shard together, no exchange.  Each rank generates its own slabs (same recipe, rank-dependent seed).
        s0, s1 = W.shard_slabs(wl, rank, world)
        my = W.Workload(f"{wl.name}_rank{rank}of{world}", wl.nx0, wl.nky0, wl.nz, wl.nv, max(s1 - s0, 1), 1, wl.kxmin,
                        wl.kymin, wl.chi_has_v, wl.seed + 1000 * rank, wl.rhs_random, wl.scale)
    else:
        # every rank owns an independent problem of the workload's shape (weak scaling)
        my = W.Workload(wl.name, wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin,
                        wl.chi_has_v, wl.seed + 1000 * rank, wl.rhs_random, wl.scale)
    chi, g, rhs = W.make_inputs(my, dev)
    nl = GeneNL(my, plane_kernel=plane_kernel)
    stream = torch.cuda.current_stream()
    warm = max(args.warmup, 3)
    w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nl.compute(chi, g, rhs, stream=stream)
    w0.record(stream)
    for _ in range(warm - 1):
        nl.compute(chi, g, rhs, stream=stream)
    w1.record(stream)
    barrier()
    steps = args.steps
    if not headline:   # side configs: at least half a second of timed work
        est = max(w0.elapsed_time(w1) / (warm - 1), 1e-3)
        steps = int(min(2000, max(args.steps, math.ceil(500.0 / est))))
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        nl.compute(chi, g, rhs, stream=stream)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item()) / steps
    if strong:
        pt = torch.tensor([float(my.planes)], dtype=torch.float64, device=dev)
        dist.all_reduce(pt, op=dist.ReduceOp.SUM)
        planes_total = int(pt.item())
    else:
        planes_total = my.planes * world
    value = planes_total / (ms_per_step * 1e-3)

    # per-kernel device time, live, with CUDA events on the launching stream
    prof_ms = {k: 0.0 for k in KERNEL_CLASSES}
    prof_n = dict.fromkeys(prof_ms, 0)
    nprof = 3
    for _ in range(nprof):
        m, n = nl.compute_profiled(chi, g, rhs, stream=stream)
        for k in prof_ms:
            prof_ms[k] += m[k]
            prof_n[k] += n[k]
    flops = per_kernel_flops(my, fused=nl.query(7) == 1.0)
    if my.chi_has_v and not prof_n.get("k_yreal") and "k_yreal" in flops and "k_ybracket" in flops:
        flops["k_ybracket"] += flops.pop("k_yreal")  # chi's y-synthesis runs inside k_ybracket_cv (no k_yreal launches)
    if "k_plane_fused" in flops and not prof_n.get("k_xinv") and not prof_n.get("k_yreal"):
        # chi per plane goes through the plane kernel itself (group kernel, CHIV): its transforms are that kernel's work
        flops["k_plane_fused"] += flops.pop("k_xinv", 0.0) + flops.pop("k_yreal", 0.0)
    fp64_model = 148 * FP64_LANES_PER_SM * 2 * 1.965e9 / 1e12
    if "probe" not in env:
        try:
            env["probe"] = gene_nl_probe_peaks()
        except Exception:  # noqa: BLE001
            env["probe"] = (None, None, None)
    probe_tf, probe_smem_gbs, _ = env["probe"]
    hbm_peak = float(env["peaks"].get("hbm_gbs", 6650.0))
    kernels = {}
    for k in prof_ms:
        if prof_n[k]:
            avg_ms = prof_ms[k] / prof_n[k]
            kernels[k] = {"launches_per_step": prof_n[k] // nprof, "ms_per_step": prof_ms[k] / nprof,
                          "avg_launch_us": 1e3 * avg_ms,
                          "tflops": flops[k] * nprof / (prof_ms[k] * 1e-3) / 1e12}
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_step"])
    # measured DRAM bytes (ncu capture of these very sources; null when the capture is older than the code)
    cap, why = measured_traffic(wl.name + ({1: "+cluster", 3: "+batched", 4: "+warp"}.get(plane_kernel, "")))
    traffic = cap[dom][0] if dom in cap else None
    traffic_step = None
    if cap and all(k in cap for k in kernels):
        # whole step: every kernel class's captured bytes per launch (average over the launches of one step of the full
        # workload) x the launches this run made per step
        traffic_step = sum(cap[k][0] * kernels[k]["launches_per_step"] for k in kernels)
    kname = plane_kernel_name(my, nl.query(7) == 1.0, nl.query(8)) if dom == "k_plane_fused" else None
    roofline = {"kernel": kname or dom, "kernel_class": dom, "bound": "alu", "achieved": kernels[dom]["tflops"], "peak": fp64_model,
                "unit": "TFLOP/s", "frac": kernels[dom]["tflops"] / fp64_model, "traffic": traffic,
                "traffic_note": why or ("ncu dram__bytes capture of one whole step (profiles/r03_dram.md), stamped with src_sha16 %s" % source_sha16()),
                "peak_source": "model 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md sect. 7)",
                "peak_measured_dfma": probe_tf, "smem_gbs_measured": probe_smem_gbs,
                "share_of_step": kernels[dom]["ms_per_step"] / sum(v["ms_per_step"] for v in kernels.values())}
    F, B = nl.query(6), nl.query(5)
    step_tf = F * my.planes / (ms_per_step * 1e-3) / 1e12
    step_gbs = B * my.planes / (ms_per_step * 1e-3) / 1e9
    t_alu, t_hbm = F / (fp64_model * 1e12), B / (hbm_peak * 1e9)
    roof_planes = 1.0 / max(t_alu, t_hbm)
    roofline_step = {"bound": "alu" if t_alu >= t_hbm else "hbm", "achieved_tflops": step_tf,
                     "achieved_hbm_gbs": step_gbs, "peak_tflops": fp64_model, "peak_hbm_gbs": hbm_peak,
                     "roofline_planes_per_s": roof_planes, "frac": (value / world) / roof_planes,
                     "frac_of_measured_dfma": (step_tf / probe_tf) if probe_tf else None,
                     "flops_per_plane": F, "bytes_per_plane": B, "algorithmic_bytes_per_step": B * my.planes,
                     "traffic_per_step": traffic_step}
    launches = nl.launches_per_compute * steps
    nl.close()

    # end to end through the host entry point: pinned host buffers, copies inside the timed region.  Arrays beyond
    # 8 GiB (configs[3]: 49 GiB of g + rhs) are represented by their first (w,s) slabs -- the host entry point streams
    # slab by slab, so the rate per plane is that of the whole array.
    e2e = None
    if do_e2e:
        nslab = my.nw * my.nspec
        slab_bytes = 2 * my.plane_bytes * my.nz * my.nv
        ns = int(max(1, min(nslab, (8 << 30) // slab_bytes)))
        sub, hchi, hg, hrhs = my, chi, g, rhs
        if ns < nslab:
            sub = W.Workload(f"{my.name}_first{ns}slabs", my.nx0, my.nky0, my.nz, my.nv, ns, 1, my.kxmin, my.kymin,
                             my.chi_has_v, my.seed, my.rhs_random, my.scale)
            hg = g.reshape((nslab,) + my.g_shape[2:])[:ns]
            hrhs = rhs.reshape((nslab,) + my.g_shape[2:])[:ns]
            hchi = chi.reshape((nslab,) + my.chi_shape[2:])[:ns]
        hchi, hg, hrhs = (t.cpu().pin_memory() for t in (hchi, hg, hrhs))
        del chi, g, rhs
        torch.cuda.empty_cache()
        with GeneNL(sub) as nlh:
            nlh.compute_host(hchi, hg, hrhs)   # warm-up (allocates staging)
            barrier()
            t0 = time.perf_counter()
            for _ in range(args.e2e_steps):
                nlh.compute_host(hchi, hg, hrhs)
            torch.cuda.synchronize()
            dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        gb = sub.plane_bytes * sub.planes
        e2e = {"value": sub.planes * world * args.e2e_steps / float(dt.item()), "unit": UNIT,
               "h2d_bytes_per_step": 2 * gb + sub.plane_bytes * sub.chi_planes, "d2h_bytes_per_step": gb,
               "steps": args.e2e_steps,
               "api": "gene_nl_compute_host (pinned host buffers)" +
                      ("" if ns == nslab else f" on the first {ns} of {nslab} (w,s) slabs = {sub.planes} planes per step") +
                      "; bound by the host link (H2D of g, rhs and chi, D2H of rhs), not by the kernels (PAPER.md:115)"}
        del hchi, hg, hrhs
    else:
        del chi, g, rhs
    torch.cuda.empty_cache()

    cpu_baseline = None
    if do_cpu and rank == 0 and world == 1:
        import oracle
        threads = oracle.num_threads()
        v, n, dt = time_oracle(wl, args.cpu_seconds / max(threads, 1), threads)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": f"{n} planes of {wl.name} (first planes, up to four (w,s) slabs), {dt:.1f} s wall"}
    return {
        "value": value, "steps": steps, "warmup": warm, "ms_per_step": ms_per_step, "scaling": "strong" if strong else "weak",
        "config": {"workload": wl.name, "configs_index": [c.name for c in W.CONFIGS].index(wl.name) if wl in W.CONFIGS else None,
                   "nx0": wl.nx0, "nky0": wl.nky0, "planes_per_gpu": my.planes,
                   "padded_grid": [wl.Nx, wl.Ny], "chi_has_v": wl.chi_has_v,
                   "cache": "inputs larger than L2 (g+rhs+chi = %.0f MiB per GPU)" %
                            ((2 * my.planes + my.chi_planes) * my.plane_bytes / 2 ** 20),
                   "parallelism": (f"one problem, (w,s) slabs sharded over {world} GPUs" if strong
                                   else f"planes x{world} (independent problems per GPU)")},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "roofline_step": roofline_step,
        "kernels": kernels, "cpu_baseline": cpu_baseline,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=None,
                    help="index into BASELINE.json configs.  Default: configs[3] (the largest single-GPU configuration: "
                         "the headline) with a per_config block for configs[1], [2], [4] measured in the same run")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="CPU work of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="headline configuration only")
    ap.add_argument("--cluster", action="store_true", help="select the cluster kernel (configs[2]-sized planes only)")
    ap.add_argument("--plane-kernel", type=int, default=None, help="gene_nl_set_plane_kernel kind (1 cluster, 2 group, 3 batched)")
    ap.add_argument("--xglobal", action="store_true",
                    help="x-global variant (SURVEY 8(f) f2): the paper's 64x16 planes, Table 4")
    ap.add_argument("--strong", action="store_true",
                    help="with --gpus N > 1: shard ONE problem's (w,s) slabs over the ranks instead of one problem per rank")
    ap.add_argument("--em", action="store_true",
                    help="chi composed on the device from phi_bar and A_par_bar (SURVEY 8(f) f1) on --config's grid")
    ap.add_argument("--xglobal-planes", type=int, default=589824, help="planes per GPU (Table 4: 589824)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    headline_idx = 3 if args.config is None else args.config
    if args.xglobal:
        xglobal_main(args)
        return
    if args.em:
        args.config = 4 if args.config is None else args.config
        em_main(args)
        return

    from paper_1310_1485_b200 import workloads as W
    wl = W.CONFIGS[headline_idx]
    if args.impl == "reference":
        reference_arm(args, wl)
        return

    import torch

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:  # noqa: BLE001
        pass
    env = {"dev": dev, "dist": dist, "world": world, "rank": rank, "local_rank": local_rank, "peaks": peaks}

    pk = None
    if args.plane_kernel is not None:
        pk = args.plane_kernel
    elif args.cluster:
        from paper_1310_1485_b200 import GENE_NL_KERNEL_CLUSTER as pk
    res = run_config(wl, args, env, do_e2e=not args.no_e2e, do_cpu=not args.no_cpu_baseline, headline=True, plane_kernel=pk)
    per_config = None
    if args.config is None and world == 1 and not args.no_per_config:
        # the other target configurations, device-resident, in the same run (same box, same clocks record)
        per_config = {}
        for idx in (1, 2, 4):
            r = run_config(W.CONFIGS[idx], args, env, do_e2e=False, do_cpu=False, headline=False)
            per_config[W.CONFIGS[idx].name] = {k: r[k] for k in ("value", "ms_per_step", "steps", "roofline",
                                                                  "roofline_step", "kernels", "clocks", "gpu_launches")}
            per_config[W.CONFIGS[idx].name]["unit"] = UNIT
        # configs[2] once more through the other kernel families (gene_nl_set_plane_kernel): the cluster kernel (Z and P
        # in distributed shared memory) and the batched kernels (Z and P through HBM scratch)
        from paper_1310_1485_b200 import GENE_NL_KERNEL_BATCHED, GENE_NL_KERNEL_CLUSTER
        for kind, label in ((GENE_NL_KERNEL_CLUSTER, "cluster kernel"), (GENE_NL_KERNEL_BATCHED, "batched kernels")):
            r = run_config(W.CONFIGS[2], args, env, do_e2e=False, do_cpu=False, headline=False, plane_kernel=kind)
            per_config[W.CONFIGS[2].name + f" (gene_nl_set_plane_kernel: {label})"] = {
                k: r[k] for k in ("value", "ms_per_step", "steps", "roofline", "roofline_step", "kernels", "clocks", "gpu_launches")}
    if per_config is not None:
        # compact summary where the driver's parsed record keeps it (inside `roofline`): every target configuration with the
        # kernel that ran, plus one device-resident line each for the x-global operator (f2) and the composed-chi operator (f1)
        def brief(r):
            return {"kernel": r["roofline"]["kernel"], "frac": r["roofline"]["frac"], "step_frac": r["roofline_step"]["frac"],
                    "ms": r["ms_per_step"], "planes_per_s": r["value"]}
        summary = {wl.name: brief(res)}
        for name, r in per_config.items():
            summary[name] = brief(r)
        extra_launches = 0
        for key, fn in (("xglobal_64x16_65536", lambda: side_xglobal(dev, peaks)), ("cfg4_em_96x48_em_composed", lambda: side_em(dev))):
            try:
                summary[key] = fn()
                extra_launches += summary[key].pop("gpu_launches", 0)
            except Exception as e:  # noqa: BLE001  (a side line must not cost the headline)
                summary[key] = {"error": str(e)[:200]}
            torch.cuda.empty_cache()
        res["roofline"]["per_config"] = summary
    if rank == 0:
        line = {
            "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": res["steps"],
            "warmup": res["warmup"], "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": res["scaling"], "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": res["config"], "clocks": res["clocks"], "e2e": res["e2e"], "gpu_launches": res["gpu_launches"],
            "roofline": res["roofline"], "roofline_step": res["roofline_step"], "kernels": res["kernels"],
            "cpu_baseline": res["cpu_baseline"],
        }
        if per_config is not None:
            line["per_config"] = per_config
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
