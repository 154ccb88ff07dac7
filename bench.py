#!/usr/bin/env python
"""bench.py - events/s per MLEM iteration of the B200 list-mode MLEM path (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one pass of the whole hot path (pre-pass, event kernel(s), finalise = one MLEM iteration, Eq. 3)
over the workload's events.  Default workload: BASELINE.json configs[1] (200x200 grid, 2.5 mm, 10^6 events,
sigma 10/40) - `cfg2` of paper_1502_07478_b200.synth; the other configs can be named with --workload.
The JSON line carries `value` (device-resident inputs, CUDA-event timing, L2 flushed between steps), `e2e`
(host buffers through jpet_mlem_iterate_host, copies inside the timed region), `roofline` for the event
kernel (ALU/SFU bound), `reconstruct` (jpet_reconstruct over the workload's iteration count:
one sort for all iterations), `cpu_baseline` (the fp64 oracle on the box's host cores)
and `clocks` sampled with nvidia-smi during the timed region.
N > 1 (torchrun): independent replicas, one per GPU ("replicas only": north_star fixes one GPU, no sharding).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/s per MLEM iteration"
UNIT = "events/s"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return json.load(open(path)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons while the timed region runs (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def summary(self):
        self.stop_flag.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower() == "active"})
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


class Ranks:
    """One process per GPU (torchrun env: RANK / LOCAL_RANK / WORLD_SIZE / MASTER_*).  Replicas only: no collective
    on the data path; the only exchanges are the barrier around the timed region and the max over ranks of its time."""

    def __init__(self, backend: str = "nccl", device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.dist = None
        self.device = device
        if self.world > 1:
            import torch.distributed as dist

            kwargs = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, **kwargs)
            self.dist = dist

    def seed(self, base: int) -> int:
        return base + self.rank                      # each replica draws its own events

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max(self, x: float) -> float:
        """Max over ranks of a host float (time of the slowest replica)."""
        if self.dist is None:
            return float(x)
        import torch

        t = torch.tensor([x], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate(self, per_rank_units: float, seconds_local: float) -> float:
        """Whole-job throughput: units processed by all ranks / time of the slowest rank."""
        return self.world * per_rank_units / self.max(seconds_local)

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


def geom(cfg):
    return (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)


def oracle_sample(cfg, events, budget_s=15.0):
    """Times the oracle as it stands on a bounded prefix of the workload (about `budget_s` of CPU work)."""
    import numpy as np

    import oracle

    cores = oracle.num_threads()
    probe = events[: min(len(events), 20000)]
    ones = np.ones((cfg.n_y, cfg.n_z))
    t0 = time.perf_counter()
    oracle.mlem_iterate(probe, *geom(cfg), ones)
    rate = len(probe) / max(time.perf_counter() - t0, 1e-6)
    n = int(min(len(events), max(20000, rate * budget_s)))
    t0 = time.perf_counter()
    _, n_evals, _ = oracle.mlem_iterate(events[:n], *geom(cfg), ones)
    dt = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"one fp64 MLEM iteration over the first {n} events of {cfg.name} ({dt:.1f} s, OpenMP over events)",
            "evals_per_s": n_evals / dt}, n, dt


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np

    import oracle
    from paper_1502_07478_b200 import synth

    per_step_budget = max(2.0, min(20.0, 120.0 / max(args.steps + args.warmup, 1)))
    events = synth.config_events(cfg, n=min(cfg.n_events, 2_000_000))
    base, n, _ = oracle_sample(cfg, events, budget_s=per_step_budget)
    ones = np.ones((cfg.n_y, cfg.n_z))
    for _ in range(args.warmup):
        oracle.mlem_iterate(events[:n], *geom(cfg), ones)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.mlem_iterate(events[:n], *geom(cfg), ones)
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    value = n / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "grid": [cfg.n_y, cfg.n_z], "pixel_mm": cfg.pixel,
                       "sigma_z": cfg.sigma_z, "sigma_dl": cfg.sigma_dl, "events_per_step": n,
                       "note": "bounded sample of the workload; time per event is constant in N (Table 1)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": base["cores"], "kind": "oracle",
                             "sample": f"one fp64 MLEM iteration over the first {n} events of {cfg.name} per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--events", type=int, default=0, help="override the number of events (0 = the config's)")
    ap.add_argument("--variant", type=int, default=-1)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--sub-tile-z", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    from paper_1502_07478_b200 import synth

    cfg = synth.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import numpy as np
    import torch

    import paper_1502_07478_b200 as jp

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    ranks = Ranks("nccl", torch.device("cuda", local_rank))
    world, rank, dist = ranks.world, ranks.rank, ranks.dist
    jp.binding.load(build_if_missing=False)
    if args.variant >= 0:
        jp.jpet_set_option("variant", args.variant)
    if args.chunk > 0:
        jp.jpet_set_option("chunk", args.chunk)
    if args.sub_tile_z > 0:
        jp.jpet_set_option("sub_tile_z", args.sub_tile_z)
    if args.ctas_per_sm > 0:
        jp.jpet_set_option("ctas_per_sm", args.ctas_per_sm)

    n_events = args.events or cfg.n_events
    events = synth.config_events(cfg, n=n_events, seed=ranks.seed(cfg.seed))     # replicas: same shape, own seed
    M = cfg.n_y * cfg.n_z
    g = geom(cfg)
    ev_d = torch.from_numpy(events).cuda()
    rho = [torch.ones(M, device="cuda"), torch.empty(M, device="cuda")]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        ranks.barrier()
        torch.cuda.synchronize()

    # ---- device-resident steps: CUDA events on the launching stream, L2 flushed between steps -------------
    def step(i, ev_pairs=None):
        src, dst = rho[i & 1], rho[(i + 1) & 1]
        if ev_pairs is None:
            jp.jpet_mlem_iterate(ev_d, *g, src, dst)
            return
        a, d = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        jp.jpet_mlem_iterate(ev_d, *g, src, dst)          # pre-pass, sort, event kernel(s), finalise: one iteration
        d.record(stream)
        ev_pairs.append((a, d))

    for i in range(args.warmup):
        step(i)
    n_evals, n_skipped = jp.jpet_get_counters()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    jp.jpet_set_option("time_kernel", 1)
    launches0 = jp.jpet_launch_count()
    pairs, kern_ms = [], []
    for i in range(args.steps):
        flush.zero_()
        step(args.warmup + i, pairs)
        ns = jp.jpet_get_option("last_kernel_ns")          # waits for this step's event kernel only
        if ns > 0:
            kern_ms.append(ns * 1e-6)
    barrier()
    launches = jp.jpet_launch_count() - launches0
    kernel_launches = jp.jpet_get_option("last_kernel_launches")     # event-kernel launches per step (one per batch)
    jp.jpet_set_option("time_kernel", 0)
    step_ms = [a.elapsed_time(d) for a, d in pairs]
    kern_ms = kern_ms or step_ms
    total_ms = ranks.max(sum(step_ms))
    ms_per_step = total_ms / args.steps
    value = world * n_events / (ms_per_step * 1e-3)

    # ---- end to end: host buffers through the C-ABI, copies inside the timed region ---------------------------
    e2e = None
    if not args.no_e2e:
        ev_h = torch.from_numpy(events).pin_memory()
        rho_h = torch.ones(M).pin_memory()
        out_h = torch.empty(M).pin_memory()
        for _ in range(2):
            jp.jpet_mlem_iterate_host(ev_h, *g, rho_h, out_h)
        barrier()
        t0 = time.perf_counter()
        k_e2e = max(3, min(args.steps, 10))
        for _ in range(k_e2e):
            jp.jpet_mlem_iterate_host(ev_h, *g, rho_h, out_h)
            rho_h, out_h = out_h, rho_h
        dt = ranks.max(time.perf_counter() - t0)
        e2e = {"value": world * n_events * k_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": int(events.nbytes + 4 * M),
               "d2h_bytes_per_step": int(4 * M), "steps": k_e2e, "ms_per_step": dt / k_e2e * 1e3,
               "timing": "host wall clock around the blocking call"}
    # ---- whole reconstruction: jpet_reconstruct sorts the events once for all iterations --------
    reconstruct = None
    if not args.no_e2e:
        n_it = max(2, cfg.n_iter)
        jp.jpet_reconstruct(ev_d, *g, rho[0], rho[1], 2)      # warm-up: allocates the buffer of the kept sorted records
        barrier()
        a, d = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        jp.jpet_reconstruct(ev_d, *g, rho[0], rho[1], n_it)
        d.record(stream)
        barrier()
        rec_ms = ranks.max(a.elapsed_time(d)) / n_it
        reconstruct = {"n_iter": n_it, "ms_per_iteration": rec_ms, "events_per_s_per_iteration": world * n_events / (rec_ms * 1e-3),
                       "note": "jpet_reconstruct: one sort for all iterations, no L2 flush between iterations"}

    clocks = sampler.summary()

    if rank != 0:
        ranks.close()
        return

    # ---- roofline of the dominant kernel (mlem_events_kernel) ---------------------------------------------
    peaks, peak_kind = measured_peaks()
    sm_mhz_peak = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    # per kernel evaluation 2 MUFU (rsqrt, ex2) at 16 MUFU lanes/clk/SM and 8 FP32
    # instructions at 128 lanes/clk/SM  ->  the SFU pipe binds at 8 evaluations/clk/SM.
    peak_evals = n_sm * 8.0 * sm_mhz_peak * 1e6
    kern_s = statistics.mean(kern_ms) * 1e-3
    achieved = n_evals / kern_s
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu --set full capture of this
    # workload (profiles/r1f_ncu_full_mlem_rows3_kernel_cfg2.txt); null for workloads without a capture
    ncu_traffic = {"cfg2": 64_319_744 + 626_432}.get(cfg.name) if n_events == cfg.n_events else None
    roofline = {"bound": "alu", "kernel": "mlem_rows3_kernel", "achieved": achieved / 1e9, "peak": peak_evals / 1e9,
                "unit": "Geval/s", "frac": achieved / peak_evals, "traffic": ncu_traffic, "traffic_unit": "bytes per launch",
                "peak_source": f"{n_sm} SMs x 16 MUFU/clk / 2 MUFU per eval x {sm_mhz_peak:.0f} MHz ({peak_kind} sm_max_mhz)",
                "kernel_ms": kern_s * 1e3, "kernel_share_of_step": statistics.mean(kern_ms) / statistics.mean(step_ms),
                "kernel_launches_per_step": kernel_launches,
                "hbm_gbs_algorithmic": (events.nbytes + 8 * M) / kern_s / 1e9, "hbm_peak_gbs": peaks.get("hbm_gbs")}

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline, _, _ = oracle_sample(cfg, events)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "grid": [cfg.n_y, cfg.n_z], "pixel_mm": cfg.pixel, "sigma_z": cfg.sigma_z,
                       "sigma_dl": cfg.sigma_dl, "events": n_events, "parallelism": "replicas only" if world > 1 else "1 gpu",
                       "l2": "flushed between steps (256 MiB memset)", "kernel_variant": jp.jpet_get_option("last_variant"),
                       "tiled": bool(jp.jpet_get_option("last_tiled")), "smem_bytes": jp.jpet_get_option("last_smem_bytes")},
            "kernel_evals_per_s": world * n_evals / (ms_per_step * 1e-3), "kernel_evals_per_iteration": n_evals,
            "px_per_event": n_evals / max(n_events, 1), "events_skipped": n_skipped,
            "e2e": e2e, "reconstruct": reconstruct, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu_baseline, "clocks": clocks}
    print(json.dumps(line))
    ranks.close()


if __name__ == "__main__":
    main()
