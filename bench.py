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


def recorded_traffic(n, state):
    """dram bytes per launch of the step kernel from the committed ncu --set full capture of the shipped kernel
    (profiles/traffic.txt, written from profiles/r02_*), if there is one for this grid and state."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        for line in open(p):
            k, _, v = line.partition(":")
            if k.strip() == f"dram_bytes_per_launch_n{n}_{state}":
                return float(v.split()[0])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons (B200_PROFILING.md), sampled every 50 ms from before the warm-up on; stop()
    keeps the samples whose time stamp falls inside the timed windows given to it (the timed steps and the second pass
    of the same steps with the per-kernel events; nvidia-smi needs ~0.3 s to start, longer than a short timed region)."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.windows = []
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def window(self, t0, t1):
        self.windows.append((t0, t1))

    def stop(self):
        import datetime
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)          # let the sample that covers the end of the last window arrive
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        rows = []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f:
            c = [t.strip() for t in line.split(",")]
            if len(c) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                sm, mx = float(c[1]), float(c[2])
            except ValueError:
                continue
            try:
                pw = float(c[3])
            except ValueError:
                pw = None
            rows.append((ts, sm, mx, pw, [nm for nm, v in zip(names, c[4:8]) if v.lower().startswith("active")]))
        self.f.close()
        os.unlink(self.f.name)
        inside = [r for r in rows if any(t0 <= r[0] <= t1 for t0, t1 in self.windows)]
        where = "timed steps + per-kernel timing pass of the same steps"
        if len(inside) < 2:       # a very short run: fall back to every sample taken under load (warm-up included)
            inside = [r for r in rows if r[3] is not None and r[3] > 400.0] or rows
            where = "all samples under load (timed region shorter than the sampling period)"
        sm = sorted(r[1] for r in inside)
        pw = sorted(r[3] for r in inside if r[3] is not None)
        reasons = sorted({nm for r in inside for nm in r[4]})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max((r[2] for r in inside), default=None),
                "power_w": pw[len(pw) // 2] if pw else None, "samples": len(sm), "window": where, "reasons": reasons}


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
def oracle_sample(cfg, n_sample, steps, warm, threads=0):
    """Time the fp64 oracle, as it stands, on a down-sized twin of the workload (same dx, density
    statistics and source density): `warm` untimed + `steps` timed steps on `threads` host threads (0 = all).
    Returns cell-updates/s."""
    from oracle import aton_oracle as orc
    from paper_1004_2503_b200 import workloads as wl
    orc.build()
    all_threads = orc.get_threads()
    orc.set_threads(threads if threads > 0 else all_threads)
    w = wl.make_config(cfg, n=n_sample)
    st, p = orc.from_workload(w)
    pos, rate = w.src_pos.numpy(), w.src_rate.numpy()
    if warm:
        orc.step(st, p, w.dt, warm, pos, rate)
    t0 = time.perf_counter()
    orc.step(st, p, w.dt, steps, pos, rate)
    dt = time.perf_counter() - t0
    used = orc.get_threads()
    orc.set_threads(all_threads)
    return n_sample ** 3 * steps / dt, dt, used


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
def timed_leg(a, do_step, dt, steps, warmup, world, stream, sampler_rank0, rewind=None):
    """W untimed + K timed steps (device time, barrier + synchronize on both sides), then K steps again with the
    library's own events around each kernel: the next K steps of the run, or -- with `rewind`, a callable that restores
    the leg's start state -- the very same W + K steps (the warm leg's state relaxes quickly: its fix-up load halves
    within tens of steps).  Returns a dict of this rank's numbers."""
    import torch
    sampler = ClockSampler(sampler_rank0) if sampler_rank0 is not None else None
    do_step(dt, warmup)
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    l0 = a.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    w0 = time.time()
    e0.record(stream)
    do_step(dt, steps)
    e1.record(stream)
    torch.cuda.synchronize()
    w1 = time.time()
    if world > 1:
        torch.distributed.barrier()
    ms_total = e0.elapsed_time(e1)
    launches = a.launch_count() - l0
    d0 = a.reduce()
    # the kernels alone: CUDA events on the library's stream around each launch (aton_set_timing), in a second pass
    # of the same K steps so the events stay out of `value`
    if rewind is not None:
        rewind()
        do_step(dt, warmup)
        torch.cuda.synchronize()
    dA = a.reduce()           # counters at the start of the second pass
    a.set_timing(True)
    w2 = time.time()
    do_step(dt, steps)
    k_ms, k_n = a.kernel_time()
    f_ms, s_ms, f_n = a.fixup_time()
    w3 = time.time()
    a.set_timing(False)
    clocks = None
    if sampler:
        sampler.window(w0, w1)
        sampler.window(w2, w3)
        clocks = sampler.stop()
    d1 = a.reduce()
    per = lambda k: (d1[k] - dA[k]) / max(steps, 1)
    return {"ms_total": ms_total, "launches": launches, "clocks": clocks, "diag": d0,
            "kernel_ms": k_ms / max(k_n, 1), "kernel_launches": k_n,
            "fixup_ms": f_ms / max(f_n, 1), "stiff_ms": s_ms / max(f_n, 1),
            "cells_redone_per_step": per("cells_subcycled"), "cells_fp64_per_step": per("cells_fp64"),
            "x_vol_end": d1["x_vol"]}


def roofline_of(leg, cells, steps, peak, peak_src, traffic, kernel_name):
    achieved = BYTES_PER_CELL_UPDATE * cells / (leg["kernel_ms"] * 1e-3) / 1e9
    step_ms = leg["ms_total"] / steps
    achieved_step = BYTES_PER_CELL_UPDATE * cells / (step_ms * 1e-3) / 1e9
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": traffic, "kernel": kernel_name, "kernel_ms": leg["kernel_ms"],
            "kernel_launches_timed": leg["kernel_launches"], "kernel_share_of_step": leg["kernel_ms"] / step_ms,
            "fixup_ms": leg["fixup_ms"], "stiff_ms": leg["stiff_ms"],
            "frac_step": achieved_step / peak, "frac_of_nominal_8TBs": achieved / 8000.0,
            "frac_step_of_nominal_8TBs": achieved_step / 8000.0,
            "target_60pct_of_8TBs_met": bool(achieved_step / 8000.0 >= 0.6),
            "algorithmic_bytes_per_launch": BYTES_PER_CELL_UPDATE * cells, "peak_source": peak_src}


def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    from paper_1004_2503_b200 import aton, build, workloads as wl
    build.build()
    cfg = args.config
    n = args.n or {1: 32, 2: 128, 3: 256, 4: 512, 5: 1024}[cfg]
    variant = 5 if args.variant is None else args.variant     # 5 = the library default
    slab_mode = args.decomp == "slab"
    if slab_mode:
        # ONE box cut into z slabs, one per rank, halo planes exchanged every step inside the library (aton_step_slab:
        # NCCL send/recv beside the interior planes, NEXT-1).
        #   --strong: THE config's box (n^3, e.g. the 1024^3 of config 5) cut N ways -> strong scaling;
        #   default:  an n x n x (n N) box, every rank generating its own n^3 part -> weak scaling.
        from paper_1004_2503_b200 import slab
        if args.strong:
            w = wl.make_config(cfg, n=n, device="cuda")               # every rank builds the same seeded box ...
            if args.flux == "hll":
                w.params["flux"] = 1
            zb, nzl = slab.slab_range(n, world, rank)                  # ... and keeps its planes
            sl = slab.SlabAton(n, n, n, w.box_cm, w.params, rank, world, native=True)
            part = [t[zb:zb + nzl].contiguous() for t in w.fields()]
            sl.set_fields(*part)
            sl.set_sources(w.src_pos.contiguous(), w.src_rate.contiguous())
            del part
            cells = float(n) * n * nzl
        else:
            w = wl.make_config(cfg, n=n, device="cuda", seed=wl.SEED_BASE + cfg + 1000 * rank)
            if args.flux == "hll":
                w.params["flux"] = 1
            sl = slab.SlabAton(n, n, n * world, w.box_cm, w.params, rank, world, native=True)
            sl.set_fields(w.nH, w.x, w.T, w.N, w.Fx, w.Fy, w.Fz)
            pos = w.src_pos.clone()
            pos[:, 2] = (pos[:, 2] + rank) / world
            sl.set_sources(pos.contiguous(), w.src_rate.contiguous())
            cells = float(n) ** 3
        a, do_step = sl.ctx, sl.step
    else:
        w = wl.make_config(cfg, n=n, device="cuda", seed=wl.SEED_BASE + cfg + 1000 * rank)
        if args.flux == "hll":          # the paper's other intercell flux; not the headline
            w.params["flux"] = 1
        if args.state == "warm":
            w = wl.synthetic_warm_state(w)
        a = aton.from_workload(w)
        a.set_kernel(variant, args.tile_y, args.tile_z)
        do_step = a.step
        cells = float(n) ** 3
    stream = torch.cuda.current_stream()

    # ---- leg 1 (the headline): device-resident timing, inputs already in HBM, aton_step only
    leg = timed_leg(a, do_step, w.dt, args.steps, args.warmup, world, stream, local_rank if rank == 0 else None)
    value, ms_per_step = aggregate(leg["ms_total"], cells * args.steps, args.steps, world)
    # the dominant kernel timed ALONE: single steps with the board left to cool for 0.7 s before each (the loop above runs
    # at the power cap and a lower SM clock; MEASURED_PEAKS' copy bandwidth is a burst figure).  Beside `frac`, not instead.
    iso_ms = None
    if rank == 0 and not slab_mode and not args.no_isolated:
        a.set_timing(True)
        best = []
        for _ in range(4):
            torch.cuda.synchronize()
            time.sleep(0.7)
            k0, n0 = a.kernel_time()
            do_step(w.dt, 1)
            k1, n1 = a.kernel_time()
            if n1 > n0:
                best.append((k1 - k0) / (n1 - n0))
        a.set_timing(False)
        iso_ms = min(best) if best else None

    # ---- end to end through the C ABI with host buffers (upload ICs, K steps, download the state)
    e2e = None
    if not args.no_e2e and not slab_mode:
        host = {k: torch.empty((n, n, n), dtype=torch.float32, pin_memory=True) for k in ("nH", "x", "T")}
        for k, src in (("nH", w.nH), ("x", w.x), ("T", w.T)):
            host[k].copy_(src)
        out = {k: torch.empty((n, n, n), dtype=torch.float32, pin_memory=True) for k in ("x", "T", "N", "Fx", "Fy", "Fz")}
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
        del host, out

    # ---- leg 2: the same grid from the synthetic warm state (fronts everywhere, ~10 % of the cells sub-cycle): what a
    #      front-dominated step costs.  Reported beside the headline, never instead of it.
    warm = None
    if not args.no_warm and not slab_mode and args.state == "dark":
        ww = wl.synthetic_warm_state(w)
        wf = [t.contiguous() for t in ww.fields()]
        del ww
        a.set_fields(*wf)
        warm_steps = min(args.steps, args.warm_steps)
        warm = timed_leg(a, do_step, w.dt, warm_steps, args.warmup, world, stream, None,
                         rewind=lambda: a.set_fields(*wf))
        del wf
        torch.cuda.empty_cache()
        warm["steps"] = warm_steps
    a.close()
    if rank != 0:
        return

    peak, peak_src = measured_hbm_peak()
    # the kernel the library launches for this grid (aton_api.cu step_kernel_of): 5 -> 4 -> 2 as the grid allows
    kvar = variant
    if kvar == 5 and not (n % 128 == 0):
        kvar = 4
    if kvar == 4 and not (n % 32 == 0):
        kvar = 2
    kname = {0: "step_ref_kernel", 2: "step_fused_kernel", 4: "step_v4_kernel", 5: "step_v5_kernel"}[kvar]
    if args.flux == "hll":
        kname = "step_hll_kernel"
        if kvar >= 4 and n % 32 == 0:
            kname = "step_hll_pk_kernel" if n % 64 == 0 else "step_hll_tiled_kernel"
    roofline = roofline_of(leg, cells, args.steps, peak, peak_src, recorded_traffic(n, "dark"), kname)
    if iso_ms:
        roofline["kernel_ms_isolated"] = iso_ms
        roofline["frac_isolated"] = BYTES_PER_CELL_UPDATE * cells / (iso_ms * 1e-3) / 1e9 / peak
        roofline["isolated"] = "best of 4 single steps, 0.7 s idle before each: the kernel alone, off the power cap"
    extra = {}
    if warm:
        extra["ms_per_step_warm"] = warm["ms_total"] / warm["steps"]
        extra["roofline_warm"] = roofline_of(warm, cells, warm["steps"], peak, peak_src, recorded_traffic(n, "warm"), kname)
        extra["state_warm"] = {"state": f"workloads.synthetic_warm_state + {args.warmup} warm-up steps, {warm['steps']} timed",
                               "x_vol_end": warm["x_vol_end"], "cells_redone_per_step": warm["cells_redone_per_step"],
                               "cells_fp64_per_step": warm["cells_fp64_per_step"], "subcycles_max": warm["diag"]["subcycles_max"]}
    cpu = None
    if not args.no_cpu:
        v, secs, cores = oracle_sample(cfg, args.cpu_sample_n, args.cpu_sample_steps, 3)
        n1 = max(32, args.cpu_sample_n // 2)
        v1, secs1, _ = oracle_sample(cfg, n1, max(4, args.cpu_sample_steps // 4), 2, threads=1)
        vw, secsw, _ = oracle_sample(2, 128, 20, 40)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs,
               "sample": f"config {cfg} twin at {args.cpu_sample_n}^3 (same dx, density statistics, source density), "
                         f"{args.cpu_sample_steps} steps after 3 warm-up, fp64, gcc -O2 + OpenMP",
               "value_1thread": v1, "seconds_1thread": secs1,
               "value_warm_cfg2": vw, "seconds_warm_cfg2": secsw,
               "sample_warm_cfg2": "config 2 on its own 128^3 grid, 20 steps after 40 oracle steps of warm-up (fronts present, "
                                   "sub-cycling live): BASELINE.md's CPU-baseline plan",
               "sample_1thread": f"the same twin at {n1}^3, {max(4, args.cpu_sample_steps // 4)} steps after 2 warm-up, one thread"}
    diag = leg["diag"]
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if (slab_mode and args.strong) else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"config {cfg}: {n}^3 periodic box, lognormal density, {int(w.src_rate.numel())} sources, "
                                   f"physics flags {dict((k, w.params[k]) for k in ('recomb_case', 'cooling', 'coll_ion', 'clump_model'))}",
                       "state": args.state + f" start + {args.warmup} warm-up steps",
                       "flux": "Lax-Friedrichs" if args.flux == "lf" else "HLL (not the headline flux)",
                       "l2": "working set per step (52 B/cell) exceeds the 126 MB L2" if 52 * cells > 4 * 126e6 else "fits in L2 (latency bound; not an HBM figure)",
                       "parallelism": (("z slabs of the one box (strong scaling)" if args.strong else "z slabs of one n x n x (n N) box")
                                       + ", halo planes exchanged every step inside the library, overlapped" if slab_mode
                                       else "replicas" if world > 1 else "single GPU"),
                       "x_vol_end": diag["x_vol"], "subcycles_per_cell_step": diag["subcycles_total"] / cells / max(diag["steps_done"], 1),
                       "subcycles_max": diag["subcycles_max"], "n_nonfinite": diag["n_nonfinite"],
                       "cells_redone_per_step": leg["cells_redone_per_step"], "cells_fp64_per_step": leg["cells_fp64_per_step"]},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": leg["launches"], "clocks": leg["clocks"]}
    line.update(extra)
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
    ap.add_argument("--strong", action="store_true", help="--decomp slab: cut the config's own box N ways (strong scaling)")
    ap.add_argument("--no-warm", action="store_true", help="skip the second (synthetic warm state) leg")
    ap.add_argument("--warm-steps", type=int, default=50, help="timed steps of the warm leg (at most --steps)")
    ap.add_argument("--flux", default="lf", choices=["lf", "hll"], help="intercell flux: Lax-Friedrichs (the headline) or HLL")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-isolated", action="store_true", help="skip the four single steps that time the step kernel alone")
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
