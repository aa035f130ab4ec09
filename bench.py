#!/usr/bin/env python
"""Benchmark of the ATON hot path: RT cell-updates/s (transport + injection + chemistry) and the
achieved fraction of the B200 HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--n 1024] [--impl ours|reference]

A "step" is one aton_step (all of SURVEY 8(a) a1-a4, a6) over the whole grid.  The default workload
is BASELINE.json's config 5 (1024^3, seeded synthetic density and sources: DESIGN.md "Input
recipe").  One process per GPU; with N > 1 (torchrun) every rank runs an independent replica of the
workload (replicas only), time = max over ranks, value = all ranks' units.
`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "RT cell-updates/sec (transport+chemistry) at 1024^3 and % of B200 HBM roofline"
UNIT = "cell-updates/s"
BYTES_PER_CELL_UPDATE = 52          # 7 fp32 reads + 6 fp32 writes
HBM_FALLBACK_GBS = 6650.0           # B200_PROFILING.md fallback


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def recorded_traffic(n):
    """dram bytes per launch of the step kernel from the committed ncu --set full capture, if any."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        for line in open(p):
            k, _, v = line.partition(":")
            if k.strip() == f"dram_bytes_per_launch_n{n}":
                return float(v.split()[0])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f:
            c = [t.strip() for t in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(value: float, world: int) -> float:
    """Max over ranks of a scalar (device time): NCCL on GPUs, gloo in the CPU tests."""
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int) -> float:
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate(local_ms_total: float, local_units: float, steps: int, world: int):
    """Whole-job throughput: all ranks' units / max-over-ranks time."""
    ms = max_over_ranks(local_ms_total, world)
    units = sum_over_ranks(local_units, world)
    return units / (ms * 1e-3), ms / max(steps, 1)


# ------------------------------------------------------------------------------------------ oracle
def oracle_sample(cfg, n_sample, steps, warm):
    """Time the fp64 oracle, as it stands, on a down-sized twin of the workload (same dx, density
    statistics and source density): `warm` untimed + `steps` timed steps.  Returns cell-updates/s."""
    from oracle import aton_oracle as orc
    from paper_1004_2503_b200 import workloads as wl
    orc.build()
    w = wl.make_config(cfg, n=n_sample)
    st, p = orc.from_workload(w)
    pos, rate = w.src_pos.numpy(), w.src_rate.numpy()
    if warm:
        orc.step(st, p, w.dt, warm, pos, rate)
    t0 = time.perf_counter()
    orc.step(st, p, w.dt, steps, pos, rate)
    dt = time.perf_counter() - t0
    return n_sample ** 3 * steps / dt, dt, orc.get_threads()


def run_reference(args, rank, world):
    if rank != 0:
        return
    n_s = args.cpu_sample_n
    per_step = max(1, args.cpu_sample_steps // max(args.steps, 1))
    total, secs, cores = 0.0, 0.0, 1
    # each bench "step" = `per_step` oracle steps on the sample; warm-up steps likewise
    v, t, cores = oracle_sample(args.config, n_s, per_step * args.steps, per_step * min(args.warmup, 3))
    total, secs = v, t
    cfg_n = args.n or {1: 32, 2: 128, 3: 256, 4: 512, 5: 1024}[args.config]
    sample = (f"config {args.config} twin at {n_s}^3 (same dx, density statistics, source density), "
              f"{per_step * args.steps} oracle steps from the dark start after {per_step * min(args.warmup, 3)} warm-up")
    line = {"impl": "reference", "metric": METRIC, "value": total, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs * 1e3 / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": f"config {args.config} ({cfg_n}^3)", "sample": sample},
            "cpu_baseline": {"value": total, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": total, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ ours
def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    from paper_1004_2503_b200 import aton, build, workloads as wl
    build.build()
    cfg = args.config
    n = args.n or {1: 32, 2: 128, 3: 256, 4: 512, 5: 1024}[cfg]
    w = wl.make_config(cfg, n=n, device="cuda", seed=wl.SEED_BASE + cfg + 1000 * rank)
    if args.state == "warm":
        w = wl.synthetic_warm_state(w)
    variant = 4 if args.variant is None else args.variant
    if args.decomp == "slab":
        # ONE box of n x n x (n * world) cells cut into z slabs, one per rank, halo planes exchanged every step
        # (NEXT-1); each rank generates its own n^3 part of the density and its sources
        from paper_1004_2503_b200 import slab
        sl = slab.SlabAton(n, n, n * world, w.box_cm, w.params, rank, world)
        sl.set_fields(w.nH, w.x, w.T, w.N, w.Fx, w.Fy, w.Fz)
        pos = w.src_pos.clone()
        pos[:, 2] = (pos[:, 2] + rank) / world
        sl.set_sources(pos.contiguous(), w.src_rate.contiguous())
        a, do_step = sl.ctx, sl.step
    else:
        a = aton.from_workload(w)
        a.set_kernel(variant, args.tile_y, args.tile_z)
        do_step = a.step
    cells = float(n) ** 3
    stream = torch.cuda.current_stream()

    # ---- device-resident timing: inputs already in HBM, aton_step only
    do_step(w.dt, args.warmup)
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = a.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    do_step(w.dt, args.steps)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    ms_total = e0.elapsed_time(e1)
    launches = a.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    diag = a.reduce()
    value, ms_per_step = aggregate(ms_total, cells * args.steps, args.steps, world)

    # ---- the dominant kernel alone: CUDA events on the library's stream around each of its launches
    #      (aton_set_timing), in a second pass of the same K steps so the events stay out of `value`
    a.set_timing(True)
    do_step(w.dt, args.steps)
    k_ms_total, k_n = a.kernel_time()
    a.set_timing(False)
    kernel_ms = k_ms_total / max(k_n, 1)

    # ---- end to end through the C ABI with host buffers (upload ICs, K steps, download the state)
    e2e = None
    if not args.no_e2e:
        host = {k: torch.empty((n, n, n), dtype=torch.float32, pin_memory=True) for k in ("nH", "x", "T")}
        for k, src in (("nH", w.nH), ("x", w.x), ("T", w.T)):
            host[k].copy_(src)
        out = {k: torch.empty((n, n, n), dtype=torch.float32, pin_memory=True) for k in ("x", "T", "N", "Fx", "Fy", "Fz")}
        del w.nH, w.x, w.T
        torch.cuda.synchronize()
        if world > 1:
            torch.distributed.barrier()
        t0 = time.perf_counter()
        a.set_fields(host["nH"], host["x"], host["T"])            # dark start: N, F = NULL
        do_step(w.dt, args.steps)
        a.get_fields(out=out)                                      # synchronises
        t_e2e = (time.perf_counter() - t0) * 1e3
        if world > 1:
            torch.distributed.barrier()
        v_e2e, _ = aggregate(t_e2e, cells * args.steps, args.steps, world)
        e2e = {"value": v_e2e, "unit": UNIT, "h2d_bytes_per_step": 3 * 4 * cells / args.steps,
               "d2h_bytes_per_step": 6 * 4 * cells / args.steps, "ms_total": t_e2e,
               "what": "aton_set_fields(host nH,x,T) + aton_step(K) + aton_get_fields(host x,T,N,F), pinned buffers"}
    a.close()
    if rank != 0:
        return

    peak, peak_src = measured_hbm_peak()
    achieved = BYTES_PER_CELL_UPDATE * cells / (kernel_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "frac_of_nominal_8TBs": achieved / 8000.0, "traffic": recorded_traffic(n),
                "kernel": {0: "step_ref_kernel", 1: "step_tiled_kernel", 2: "step_fused_kernel", 3: "step_v3_kernel", 4: "step_v4_kernel"}[variant],
                "kernel_ms": kernel_ms, "kernel_launches_timed": k_n,
                "kernel_share_of_step": kernel_ms / (ms_total / args.steps), "algorithmic_bytes_per_launch": BYTES_PER_CELL_UPDATE * cells,
                "peak_source": peak_src}
    cpu = None
    if not args.no_cpu:
        v, secs, cores = oracle_sample(cfg, args.cpu_sample_n, args.cpu_sample_steps, 3)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs,
               "sample": f"config {cfg} twin at {args.cpu_sample_n}^3 (same dx, density statistics, source density), "
                         f"{args.cpu_sample_steps} steps after 3 warm-up, fp64, gcc -O2 + OpenMP"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"config {cfg}: {n}^3 periodic box, lognormal density, {int(w.src_rate.numel())} sources, "
                                   f"physics flags {dict((k, w.params[k]) for k in ('recomb_case', 'cooling', 'coll_ion', 'clump_model'))}",
                       "state": args.state + f" start + {args.warmup} warm-up steps",
                       "l2": "working set per step (52 B/cell) exceeds the 126 MB L2" if 52 * cells > 4 * 126e6 else "fits in L2 (latency bound; not an HBM figure)",
                       "parallelism": ("z slabs of one box, halo planes exchanged every step" if args.decomp == "slab"
                                       else "replicas" if world > 1 else "single GPU"),
                       "x_vol_end": diag["x_vol"], "subcycles_per_cell_step": diag["subcycles_total"] / cells / max(diag["steps_done"], 1),
                       "subcycles_max": diag["subcycles_max"], "n_nonfinite": diag["n_nonfinite"]},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--n", type=int, default=None, help="grid size override (down-sized twin)")
    ap.add_argument("--state", default="dark", choices=["dark", "warm"])
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default, the north_star's single-GPU path) or z slabs of one box")
    ap.add_argument("--variant", type=int, default=None)
    ap.add_argument("--tile-y", type=int, default=0)
    ap.add_argument("--tile-z", type=int, default=0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-sample-n", type=int, default=128)
    ap.add_argument("--cpu-sample-steps", type=int, default=100)
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        import torch
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl")
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
