#!/usr/bin/env python
"""bench.py - events/s per MLEM iteration of the B200 list-mode MLEM path (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl reference] [--sweep] [--microbench]

A "step" is one pass of the whole hot path (pre-pass, sort, event kernels, finalise = one MLEM iteration, Eq. 3) over the
workload's events through one jpet_mlem_iterate call.  Default workload: BASELINE.json configs[4], the largest
single-GPU configuration (512x512 grid of 1 mm, 10^8 events in 10 internal batches of 10^7, sigma 10/40) - `cfg5` of
paper_1502_07478_b200.synth.  The events are drawn on the device with jpet_generate_events (the recipe of DESIGN.md
section 5 with a counter-based generator; seeded), so the default run takes minutes, not the tens of minutes numpy needs
for 10^8 events.  The JSON line carries
  value        device-resident inputs, CUDA-event timing on the launching stream, L2 flushed between steps
  e2e          host buffers through jpet_mlem_iterate_host, host<->device copies inside the timed region
  roofline     the tiled event kernel (ALU/SFU bound), timed live with CUDA events
  per_config   the same measurement for the other four BASELINE configs and the paper-shaped workload fig4
  reconstruct  jpet_reconstruct over several iterations (one sort for all of them)
  histogram    jpet_direct_histogram (Eq. 2 + binning) over the workload's events against the HBM roofline
  cpu_baseline the fp64 oracle on the box's host cores (all cores and one thread), bounded sample
  clocks       nvidia-smi samples during the timed region
N > 1 (torchrun): the events are sharded over the ranks (paper_1502_07478_b200.sharding: every rank accumulates its own
events, the accumulators are summed, every rank finalises); per-GPU work is fixed ("scaling": "weak").
--sweep: N = 10 ... 100 x 10^6 events on the paper's own set-up (fig4; Table 1): time per iteration / N.
--microbench: builds and runs bench_micro.cu (FFMA / MUFU / red.global.add / shared-memory RMW peaks).
"""
from __future__ import annotations

import argparse
import hashlib
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
DEFAULT_WORKLOAD = "cfg5"


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
    """One process per GPU (torchrun env: RANK / LOCAL_RANK / WORLD_SIZE / MASTER_*): the barrier around the timed region,
    the max over ranks of its time, and the process group the sharded iteration reduces over."""

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
        return base + self.rank                      # each rank draws its own shard of the event list

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max(self, x: float) -> float:
        """Max over ranks of a host float (time of the slowest rank)."""
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


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(cfg, events, budget_s=12.0, one_thread_budget_s=5.0):
    """Times the oracle as it stands on a bounded prefix of the workload: all host cores (about `budget_s` of CPU work) and
    one thread (SURVEY.md 8(d) "Oracle timing")."""
    import numpy as np

    import oracle

    cores = oracle.num_threads()
    probe = events[: min(len(events), 5000)]
    ones = np.ones((cfg.n_y, cfg.n_z))
    t0 = time.perf_counter()
    oracle.mlem_iterate(probe, *geom(cfg), ones)
    rate = len(probe) / max(time.perf_counter() - t0, 1e-6)
    n = int(min(len(events), max(5000, rate * budget_s)))
    t0 = time.perf_counter()
    _, n_evals, _ = oracle.mlem_iterate(events[:n], *geom(cfg), ones)
    dt = time.perf_counter() - t0
    n1 = int(min(n, max(1000, rate / max(cores, 1) * one_thread_budget_s)))
    t0 = time.perf_counter()
    oracle.mlem_iterate(events[:n1], *geom(cfg), ones, n_threads=1)
    dt1 = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": cores, "cpu": cpu_model(), "kind": "oracle",
            "sample": f"one fp64 MLEM iteration over the first {n} events of {cfg.name} ({dt:.1f} s, OpenMP over events)",
            "evals_per_s": n_evals / dt,
            "one_thread": {"value": n1 / dt1, "unit": UNIT, "sample": f"the first {n1} events, 1 thread ({dt1:.1f} s)"}}, n, dt


def host_events(cfg, n, seed=None):
    """Events for the oracle legs (no GPU needed): the numpy recipe of synth.py."""
    from paper_1502_07478_b200 import synth

    return synth.config_events(cfg, n=n, seed=seed)


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np

    import oracle

    per_step_budget = max(2.0, min(15.0, 100.0 / max(args.steps + args.warmup, 1)))
    events = host_events(cfg, min(cfg.n_events, 400_000))
    base, n, _ = oracle_sample(cfg, events, budget_s=per_step_budget, one_thread_budget_s=2.0)
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
                       "sigma_z": cfg.sigma_z, "sigma_dl": cfg.sigma_dl, "events": args.events or cfg.n_events,
                       "sample_events": n,
                       "note": "each step is a bounded sample of the workload's events; time per event is constant in N (Table 1)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": base["cores"], "cpu": base["cpu"], "kind": "oracle",
                             "sample": f"one fp64 MLEM iteration over the first {n} events of {cfg.name} per step",
                             "one_thread": base["one_thread"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_microbench():
    exe = os.path.join(ROOT, "gpurun_out", "bench_micro")
    os.makedirs(os.path.dirname(exe), exist_ok=True)
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe, os.path.join(ROOT, "bench_micro.cu")],
                   check=True)
    subprocess.run([exe], check=True)


# ------------------------------------------------------------------------------------------------------------------
class Device:
    """What one measurement needs: the library, torch, the stream, an L2 flush buffer."""

    def __init__(self, local_rank):
        import torch

        import paper_1502_07478_b200 as jp

        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        torch.cuda.set_device(local_rank)
        jp.binding.load(build_if_missing=False)
        self.torch, self.jp, self.local_rank = torch, jp, local_rank
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
        self.stream = torch.cuda.current_stream()
        self.n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count

    def events(self, cfg, n, seed):
        ev = self.torch.empty((n, 3), device="cuda")
        self.jp.jpet_generate_events(cfg.phantom, n, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, seed, ev)
        return ev


def measure(dev: Device, ranks: Ranks, cfg, ev_d, steps, warmup, sharded=None):
    """W warm-up + K timed steps of one MLEM iteration over ev_d; CUDA events on the launching stream around every step,
    the event-kernel launches timed inside the library ("time_kernel"), L2 flushed between steps."""
    torch, jp = dev.torch, dev.jp
    M = cfg.n_y * cfg.n_z
    g = geom(cfg)
    rho = [torch.ones(M, device="cuda"), torch.empty(M, device="cuda")]

    def iterate(src, dst):
        if sharded is not None:
            sharded.iterate(ev_d, g, src, dst)
        else:
            jp.jpet_mlem_iterate(ev_d, *g, src, dst)

    if warmup + steps < 1:
        raise ValueError("measure() needs at least one iteration (warmup + steps >= 1)")
    for i in range(warmup):
        iterate(rho[i & 1], rho[(i + 1) & 1])
    torch.cuda.synchronize()
    ranks.barrier()
    torch.cuda.synchronize()
    jp.jpet_set_option("time_kernel", 1)
    launches0 = jp.jpet_launch_count()
    pairs, kern_ms = [], []
    for i in range(steps):
        dev.flush.zero_()
        a, d = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(dev.stream)
        iterate(rho[(warmup + i) & 1], rho[(warmup + i + 1) & 1])     # pre-pass, sort, event kernel(s), finalise
        d.record(dev.stream)
        pairs.append((a, d))
        ns = jp.jpet_get_option("last_kernel_ns")                      # waits for this step's event kernels only
        if ns > 0:
            kern_ms.append(ns * 1e-6)
    torch.cuda.synchronize()
    ranks.barrier()
    torch.cuda.synchronize()
    launches = jp.jpet_launch_count() - launches0
    n_evals, n_skipped = jp.jpet_get_counters()                       # of the last iteration run (every iteration counts the same)
    kernel_launches = jp.jpet_get_option("last_kernel_launches")      # event-kernel launches per step (one per batch)
    jp.jpet_set_option("time_kernel", 0)
    step_ms = [a.elapsed_time(d) for a, d in pairs]
    kern_ms = kern_ms or step_ms
    plan = jp.jpet_plan_describe(*g)
    return {"step_ms_sum": sum(step_ms), "step_ms": statistics.mean(step_ms), "kern_ms": statistics.mean(kern_ms),
            "n_evals": n_evals, "n_skipped": n_skipped, "launches": int(launches), "kernel_launches": int(kernel_launches),
            "plan": plan, "shape": shape_names(jp),
            "tiled": bool(jp.jpet_get_option("last_tiled")), "smem": jp.jpet_get_option("last_smem_bytes")}


def roofline_of(dev: Device, cfg, n_events, m, peaks, peak_kind):
    """The tiled event kernel against its bounds.  `frac` is against the ALGORITHMIC SFU peak
    (2 MUFU per kernel evaluation), the figure that stays comparable across rounds; `bounds` lists what
    can bind the kernel as it runs."""
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    clk = sm_mhz * 1e6
    deg = m["plan"]["degree"] if m["tiled"] else 0
    mufu_as_run = 1 if deg > 0 else 2
    peak_alg = dev.n_sm * 16.0 / 2.0 * clk                          # 16 MUFU lanes / clk / SM, 2 MUFU per evaluation
    peak_run = dev.n_sm * 16.0 / mufu_as_run * clk
    peak_smem = dev.n_sm * 128.0 / 12.0 * clk                       # 128 B / clk / SM of shared memory, 3 x 4 B per evaluation
    kern_s = m["kern_ms"] * 1e-3
    achieved = m["n_evals"] / kern_s
    M = cfg.n_y * cfg.n_z
    batches = max(1, m["kernel_launches"])
    algorithmic = (12.0 * n_events + 8.0 * M) / batches            # bytes per launch: 12 B / event + 8 B / pixel per iteration
    # what the kernel moves per launch by construction: the 64-byte records the sort wrote, w staged and the regions flushed
    # once per work item (sub-tile + halo), the accumulator image read-modify-written in L2
    p = m["plan"]
    items = n_events / batches / max(p["chunk"], 1) + (cfg.n_y + 2 * p["Hy"]) / max(p["Sy"], 1) * (cfg.n_z + 2 * p["Hz"]) / max(p["Sz"], 1)
    model = 64.0 * n_events / batches + 8.0 * M
    l2_model = items * p["HS"] * p["WZ"] * 4.0 * (1 + p["groups_per_cta"])
    measured = ncu_traffic(cfg.name, n_events, batches)
    bounds = {"sfu_algorithmic_2_mufu_per_eval": peak_alg / 1e9, "sfu_as_run": peak_run / 1e9, "mufu_per_eval_as_run": mufu_as_run,
              "shared_memory_12_B_per_eval": peak_smem / 1e9, "unit": "Geval/s"}
    binding = min(peak_run, peak_smem)
    return {"bound": "alu", "kernel": "mlem_rows_kernel<" + m["shape"] + ">", "achieved": achieved / 1e9, "peak": peak_alg / 1e9,
            "unit": "Geval/s", "frac": achieved / peak_alg,
            "peak_source": f"{dev.n_sm} SMs x 16 MUFU/clk / 2 MUFU per eval (algorithmic, SURVEY.md 8(d)) x {sm_mhz:.0f} MHz ({peak_kind} sm_max_mhz)",
            "bounds": bounds, "binding_bound": "shared_memory_12_B_per_eval" if peak_smem < peak_run else "sfu_as_run",
            "frac_of_binding_bound": achieved / binding,
            "traffic": measured, "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
            "traffic_source": "profiles/r2_traffic.json: an ncu --set full capture of commit a2db65d, NOT re-measured by this run; "
                              "null when csrc/mlem_rows.cuh has changed since that capture",
            "bound_note": "bound / peak / frac are the ALGORITHMIC SFU roofline of SURVEY.md 8(d) (2 MUFU per evaluation), kept so "
                          "that rounds stay comparable; what limits the kernel as it runs is binding_bound / frac_of_binding_bound",
            "traffic_model": model, "traffic_model_note": "64 B record read per event + 8 B per pixel; the shared-memory regions move "
            f"{l2_model / 1e6:.0f} MB per launch through L2",
            "algorithmic_bytes": algorithmic, "traffic_over_algorithmic": (measured or model) / algorithmic,
            "kernel_ms": m["kern_ms"], "kernel_share_of_step": m["kern_ms"] / m["step_ms"],
            "kernel_launches_per_step": m["kernel_launches"],
            "hbm_gbs_algorithmic": algorithmic * batches / kern_s / 1e9, "hbm_peak_gbs": peaks.get("hbm_gbs")}


def shape_names(jp):
    """Shape of the last iteration's event kernel; "a + b" when the sort made two degree classes (b walks the events whose own
    truncation bound allows the degree-3 exponent polynomial)."""
    name = jp.jpet_shape_name(jp.jpet_get_option("last_variant"))
    low = jp.jpet_get_option("last_variant_low")
    return name + (" + " + jp.jpet_shape_name(low) if low >= 0 else "")


def ncu_traffic(name, n_events, batches):
    """dram bytes per launch of the event kernel from the committed ncu --set full captures (profiles/r2_traffic.json:
    bytes per event of one launch, measured; null when the workload has no capture)."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.json")
    try:
        rec = json.load(open(path))
        per_event = rec["dram_bytes_per_event"].get(name)
        # a profiler figure read from a committed file, not measured by this run: only valid for the kernel it was taken on
        src = open(os.path.join(ROOT, rec["kernel_source"]), "rb").read()
        if hashlib.sha256(src).hexdigest()[:16] != rec["kernel_source_sha256_16"]:
            return None
    except Exception:
        return None
    return None if per_event is None else per_event * n_events / batches


def run_sweep(dev: Device, ranks: Ranks, args):
    """Table 1: time of one iteration against the number of events, N = 10 ... 100 x 10^6, on the paper's
    own set-up (fig4: R = 130, L = 300, 4 mm pixels, Table 2 phantom).  The paper's point is that time / N is constant."""
    from paper_1502_07478_b200 import synth

    cfg = synth.CONFIGS["fig4"]
    ev_all = dev.events(cfg, 100_000_000, ranks.seed(cfg.seed + 1000))
    rows = []
    for n in range(10_000_000, 100_000_001, 10_000_000):
        m = measure(dev, ranks, cfg, ev_all[:n], max(2, min(args.steps, 5)), 3)
        rows.append({"events": n, "ms_per_iteration": m["step_ms"], "ns_per_event": m["step_ms"] * 1e6 / n,
                     "events_per_s": n / (m["step_ms"] * 1e-3)})
    per = [r["ns_per_event"] for r in rows]
    line = {"sweep": "Table 1 (PAPER.md:187-198) on fig4", "rows": rows, "ns_per_event_mean": statistics.mean(per),
            "ns_per_event_spread": (max(per) - min(per)) / statistics.mean(per),
            "paper_context": {"GTX 770": "4.72 s per 10^8 events (47 ns/event)", "Xeon E5-1650 v2, 6 cores": "118 s per 10^8 events",
                              "note": "other hardware, workload size not stated: context only"}}
    if ranks.rank == 0:
        print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--events", type=int, default=0, help="override the number of events (0 = the config's)")
    ap.add_argument("--variant", type=int, default=-1)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--ctas-per-sm", type=int, default=0)
    ap.add_argument("--sub-tile-z", type=int, default=0)
    ap.add_argument("--shard-mode", default="p2p", choices=["p2p", "nccl"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--host-events", action="store_true", help="draw the events with the numpy recipe (synth.py) instead of the device generator")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--microbench", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    from paper_1502_07478_b200 import synth

    cfg = synth.CONFIGS[args.workload]
    if args.microbench:
        run_microbench()
        return
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import numpy as np
    import torch

    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dev = Device(local_rank)
    jp = dev.jp
    ranks = Ranks("nccl", torch.device("cuda", local_rank))
    world, rank = ranks.world, ranks.rank
    for name, val in (("variant", args.variant if args.variant >= 0 else None), ("chunk", args.chunk or None),
                      ("sub_tile_z", args.sub_tile_z or None), ("ctas_per_sm", args.ctas_per_sm or None)):
        if val is not None:
            jp.jpet_set_option(name, val)
    if args.sweep:
        run_sweep(dev, ranks, args)
        ranks.close()
        return

    n_events = args.events or cfg.n_events
    if args.host_events:
        ev_d = torch.from_numpy(host_events(cfg, n_events, ranks.seed(cfg.seed))).cuda()
        data = "synthetic (numpy recipe of synth.py, seeded)"
    else:
        ev_d = dev.events(cfg, n_events, ranks.seed(cfg.seed))       # every rank: its own shard of a world x n_events list
        data = "synthetic (jpet_generate_events on the device: recipe of DESIGN.md section 5, Philox4x32-10, seeded)"
    M = cfg.n_y * cfg.n_z
    g = geom(cfg)
    sharded = None
    if world > 1:
        from paper_1502_07478_b200.sharding import ShardedMlem

        sharded = ShardedMlem(ranks.dist, mode=args.shard_mode)

    sampler = ClockSampler(local_rank)
    sampler.start()
    m = measure(dev, ranks, cfg, ev_d, args.steps, args.warmup, sharded)
    clocks = sampler.summary()
    total_ms = ranks.max(m["step_ms_sum"])
    ms_per_step = total_ms / args.steps
    value = world * n_events / (ms_per_step * 1e-3)

    # ---- end to end: host buffers through the C-ABI, copies inside the timed region ---------------------------
    e2e = None
    if not args.no_e2e and world == 1:
        ev_h = torch.empty((n_events, 3), dtype=torch.float32).pin_memory()
        ev_h.copy_(ev_d)
        rho_h = torch.ones(M).pin_memory()
        out_h = torch.empty(M).pin_memory()
        for _ in range(2):
            jp.jpet_mlem_iterate_host(ev_h, *g, rho_h, out_h)
        t0 = time.perf_counter()
        k_e2e = max(3, min(args.steps, 5))
        for _ in range(k_e2e):
            jp.jpet_mlem_iterate_host(ev_h, *g, rho_h, out_h)
            rho_h, out_h = out_h, rho_h
        dt = time.perf_counter() - t0
        e2e = {"value": n_events * k_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": int(ev_h.numel() * 4 + 4 * M),
               "d2h_bytes_per_step": int(4 * M), "steps": k_e2e, "ms_per_step": dt / k_e2e * 1e3,
               "timing": "host wall clock around the blocking call jpet_mlem_iterate_host (pinned host buffers)"}
        del ev_h
    elif not args.no_e2e:
        e2e = {"value": None, "unit": UNIT, "note": "measured at 1 GPU only (the host-buffer call is single-device)"}

    # ---- whole reconstruction: jpet_reconstruct sorts the events once for all iterations --------
    reconstruct = None
    histogram = None
    if world == 1 and not args.no_e2e:
        n_it = 3 if n_events > 20_000_000 else max(2, min(cfg.n_iter, 10))
        n_rec = min(n_events, 30_000_000)                              # the kept records are 64 B per event
        rho = [torch.ones(M, device="cuda"), torch.empty(M, device="cuda")]
        jp.jpet_reconstruct(ev_d[:n_rec], *g, rho[0], rho[1], 2)       # warm-up: allocates the buffer of the kept sorted records
        torch.cuda.synchronize()
        a, d = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(dev.stream)
        jp.jpet_reconstruct(ev_d[:n_rec], *g, rho[0], rho[1], n_it)
        d.record(dev.stream)
        torch.cuda.synchronize()
        rec_ms = a.elapsed_time(d) / n_it
        reconstruct = {"n_iter": n_it, "events": n_rec, "ms_per_iteration": rec_ms, "events_per_s_per_iteration": n_rec / (rec_ms * 1e-3),
                       "note": "jpet_reconstruct: one sort for all iterations, no L2 flush between iterations"}
        jp.jpet_release()                                              # frees the kept records (1.9 GB at 3x10^7 events)
        # ---- direct reconstruction histogram (Eq. 2 + binning, Fig. 4b): HBM-bound companion kernel -----------
        hist = torch.zeros(M, dtype=torch.int32, device="cuda")
        for _ in range(3):
            jp.jpet_direct_histogram(ev_d, cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel, hist, count_outside=False)
        torch.cuda.synchronize()
        hs = []
        for _ in range(5):
            dev.flush.zero_()
            a, d = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(dev.stream)
            jp.jpet_direct_histogram(ev_d, cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel, hist, count_outside=False)
            d.record(dev.stream)
            torch.cuda.synchronize()
            hs.append(a.elapsed_time(d))
        h_ms = statistics.mean(hs)

    if rank != 0:
        ranks.close()
        return

    peaks, peak_kind = measured_peaks()
    roofline = roofline_of(dev, cfg, n_events, m, peaks, peak_kind)
    if world == 1 and not args.no_e2e:
        gbs = 12.0 * n_events / (h_ms * 1e-3) / 1e9
        histogram = {"kernel": "direct_histogram_kernel", "events": n_events, "ms": h_ms, "events_per_s": n_events / (h_ms * 1e-3),
                     "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                                  "frac": gbs / float(peaks.get("hbm_gbs", 6650.0)), "algorithmic_bytes_per_event": 12}}

    # ---- the other configs of BASELINE.json and the paper-shaped workload, same measurement, fewer steps -------
    per_config = None
    if not args.no_per_config and world == 1 and args.workload == DEFAULT_WORKLOAD and not args.events:
        per_config = {}
        del ev_d
        torch.cuda.empty_cache()
        for name in ("cfg1", "cfg2", "cfg3", "cfg4", "fig4"):
            c = synth.CONFIGS[name]
            ev_c = dev.events(c, c.n_events, c.seed)
            mc = measure(dev, ranks, c, ev_c, 5, 3)
            rc = roofline_of(dev, c, c.n_events, mc, peaks, peak_kind)
            per_config[name] = {"value": c.n_events / (mc["step_ms"] * 1e-3), "unit": UNIT, "ms_per_step": mc["step_ms"], "events": c.n_events,
                                "grid": [c.n_y, c.n_z], "kernel_evals_per_s": mc["n_evals"] / (mc["step_ms"] * 1e-3),
                                "px_per_event": mc["n_evals"] / c.n_events, "kernel": rc["kernel"], "kernel_ms": rc["kernel_ms"],
                                "roofline_frac": rc["frac"], "frac_of_binding_bound": rc["frac_of_binding_bound"], "steps": 5}
            del ev_c

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline, _, _ = oracle_sample(cfg, host_events(cfg, min(cfg.n_events, 1_500_000)))

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": data,
            "config": {"workload": cfg.name, "grid": [cfg.n_y, cfg.n_z], "pixel_mm": cfg.pixel, "sigma_z": cfg.sigma_z,
                       "sigma_dl": cfg.sigma_dl, "events": n_events, "events_per_gpu": n_events,
                       "parallelism": (f"events sharded over {world} GPUs, accumulators summed ({args.shard_mode})" if world > 1 else "1 gpu"),
                       "batches": m["kernel_launches"], "l2": "flushed between steps (256 MiB memset)", "kernel_shape": m["shape"],
                       "tiled": m["tiled"], "smem_bytes": m["smem"]},
            "kernel_evals_per_s": world * m["n_evals"] / (ms_per_step * 1e-3), "kernel_evals_per_iteration": m["n_evals"],
            "px_per_event": m["n_evals"] / max(n_events, 1), "events_skipped": m["n_skipped"],
            "e2e": e2e, "reconstruct": reconstruct, "histogram": histogram, "gpu_launches": m["launches"], "roofline": roofline,
            "per_config": per_config, "cpu_baseline": cpu_baseline, "clocks": clocks}
    print(json.dumps(line))
    ranks.close()


if __name__ == "__main__":
    main()
