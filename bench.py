#!/usr/bin/env python
"""bench.py — the ARGUS hot path on B200: raw kernel events -> per-(rank, step, sig) summaries and
spans -> cross-rank median/MAD diagnosis (BASELINE.json `metric`), on seeded synthetic events.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload production] [--impl ours|reference]

One step = one pass of the whole path over the workload: argus_reset + argus_aggregate +
argus_phase_times + argus_diagnose.  `value` is timed with CUDA events with the events resident in
HBM; `e2e` is the same step through argus_aggregate_host with HOST (pinned) buffers: the 256 MiB
chunked host->device copies and the device->host read of the diagnosis are inside the timed region.
Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle (oracle/) instead.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "kernel events/s and raw-event GB/s (fraction of B200 HBM peak), bit-exact"
CHUNK_EVENTS = 8 * 1024 * 1024          # 256 MiB of 32-byte records (BASELINE.json configs[4])
RING_SLOTS = 3


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def profile_traffic_bytes(workload: str):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, or None."""
    p = os.path.join(ROOT, "profiles", f"{workload}_seg_traffic.txt")
    try:
        with open(p) as f:
            for line in f:
                if line.startswith("traffic_bytes_per_launch"):
                    return float(line.split("=")[1])
    except Exception:
        pass
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks"}

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.err = None

    def run(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
            while not self._stop_evt.is_set():
                self.samples.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                try:
                    bits = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    bits = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
                time.sleep(0.02)
        except Exception as e:  # NVML missing: report it, do not fail the bench
            self.err = repr(e)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        out = {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
               "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.err:
            out["error"] = self.err
        return out


# ---------------------------------------------------------------------------------------------
def oracle_sample(wl, n_ranks_sample: int, threads: int):
    """Time the oracle, as it stands, on the first `n_ranks_sample` ranks of the workload."""
    from oracle import Oracle
    s = wl.spec
    if s.shuffle:
        ev = wl.expand_host(0, s.n_ranks, threads=threads)
        ev = ev[: n_ranks_sample * s.n_steps * s.n_events]
        R = s.n_ranks
    else:
        ev = wl.expand_host(0, n_ranks_sample, threads=threads)
        R = n_ranks_sample
    o = Oracle(R, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    t0 = time.perf_counter()
    o.aggregate(ev)
    o.phase_times()
    o.diagnose()
    dt = time.perf_counter() - t0
    return ev.size, dt


def run_reference(args, world):
    """--impl reference: the CPU oracle on this box's host cores (rank 0 only)."""
    from paper_2606_20374_b200.workload import build_workload
    if world.rank != 0:
        return
    wl = build_workload(args.workload)
    s = wl.spec
    sample_ranks = max(1, min(s.n_ranks, (8_000_000 // (s.n_steps * s.n_events)) or 1))
    threads = os.cpu_count() or 1
    times, n_ev = [], 0
    for i in range(args.warmup + args.steps):
        n_ev, dt = oracle_sample(wl, sample_ranks, threads)
        if i >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    v = n_ev / t
    sample = f"first {sample_ranks} of {s.n_ranks} ranks ({n_ev} events) of '{s.name}' per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": s.name, "n_ranks": s.n_ranks, "n_steps": s.n_steps,
                   "events_per_rank_step": s.n_events, "n_sigs": s.n_sigs, "n_phases": s.n_phases},
        "raw_event_gbs": 32 * v / 1e9,
        "cpu_baseline": {"value": v, "unit": "events/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ---------------------------------------------------------------------------------------------
def run_ours(args, world):
    import torch
    from paper_2606_20374_b200 import argus as A
    from paper_2606_20374_b200 import dist as D
    from paper_2606_20374_b200.workload import build_workload
    import dataclasses

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(world.local_rank)
    dev = world.local_rank
    wl0 = build_workload(args.workload)
    spec = dataclasses.replace(wl0.spec, seed=D.job_seed(wl0.spec.seed, world))
    wl = build_workload(spec) if world.rank else wl0
    s = wl.spec
    n = s.total_events

    d_ev = wl.expand_device(device=f"cuda:{dev}")
    ctx = A.Argus(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base, sorted_hint=not s.shuffle, device=dev)
    if args.variant:
        ctx.tune(A.TUNE_SEG_VARIANT, args.variant)
    rec = ctx.alloc_records()
    outs = ctx.alloc_diag()
    torch.cuda.synchronize()

    def step(ev_pairs=None):
        ctx.reset(rec)
        if ev_pairs is not None:
            ev_pairs[0].record()
        ctx.aggregate(d_ev, n, rec)
        if ev_pairs is not None:
            ev_pairs[1].record()
        ctx.phase_times(rec)
        ctx.diagnose(rec, outs)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    D.barrier(world)

    sampler = ClockSampler(dev)
    sampler.start()
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    torch.cuda.synchronize()
    t_beg.record()
    for i in range(args.steps):
        step(pairs[i])
    t_end.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    D.barrier(world)
    ms_total = D.max_over_ranks(world, t_beg.elapsed_time(t_end))
    ms_step = ms_total / args.steps
    agg_ms = float(np.mean([a.elapsed_time(b) for a, b in pairs]))
    n_valid, n_invalid = ctx.stats()
    total_events = D.sum_over_ranks(world, float(n))
    value = total_events / (ms_step * 1e-3)

    # ---- e2e: HOST buffers through argus_aggregate_host, copies inside the timed region ----------
    e2e = None
    if not args.no_e2e:
        try:
            h_ev = torch.empty(n * 32, dtype=torch.uint8, pin_memory=True)
            h_ev.copy_(d_ev)
            torch.cuda.synchronize()
            del d_ev
            chunk = min(CHUNK_EVENTS, n)
            d_ring = torch.empty(RING_SLOTS * chunk * 32, dtype=torch.uint8, device=f"cuda:{dev}")
            h_out = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True) for k, v in outs.items()}
            d2h = sum(v.numel() * v.element_size() for v in outs.values())

            def e2e_step():
                ctx.reset(rec)
                ctx.aggregate_host(h_ev, n, chunk, d_ring, RING_SLOTS, rec)
                ctx.phase_times(rec)
                ctx.diagnose(rec, outs)
                for k in outs:
                    h_out[k].copy_(outs[k], non_blocking=True)

            e2e_steps = max(1, min(args.steps, args.e2e_steps))
            e2e_step()
            torch.cuda.synchronize()
            D.barrier(world)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(e2e_steps):
                e2e_step()
            b.record()
            torch.cuda.synchronize()
            e_ms = D.max_over_ranks(world, a.elapsed_time(b)) / e2e_steps
            e2e = {"value": total_events / (e_ms * 1e-3), "unit": "events/s", "ms_per_step": e_ms,
                   "steps": e2e_steps, "h2d_bytes_per_step": 32 * n, "d2h_bytes_per_step": d2h,
                   "h2d_gbs": 32 * n / (e_ms * 1e-3) / 1e9, "chunk_bytes": chunk * 32,
                   "ring_slots": RING_SLOTS}
        except Exception as e:  # e.g. the box cannot pin the whole buffer
            e2e = {"value": None, "unit": "events/s", "error": repr(e)[:200],
                   "h2d_bytes_per_step": 32 * n, "d2h_bytes_per_step": None}

    if world.rank != 0:
        return
    peak, peak_src = measured_peak_gbs()
    alg_bytes = 32 * n + ctx.table_bytes          # raw bytes read + summary bytes written (NS)
    achieved = alg_bytes / (agg_ms * 1e-3) / 1e9
    traffic = profile_traffic_bytes(s.name)
    diag_bytes = 8 * s.n_ranks * s.n_steps * s.n_sigs + s.n_ranks * s.n_steps * (s.n_sigs + s.n_phases + 1) \
        + 32 * s.n_steps * (s.n_sigs + s.n_phases + 1)
    step_bytes = alg_bytes + diag_bytes
    out = {
        "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world.size, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": s.name, "n_ranks": s.n_ranks, "n_steps": s.n_steps,
                   "events_per_rank_step": s.n_events, "n_sigs": s.n_sigs, "n_phases": s.n_phases,
                   "events": n, "raw_bytes": 32 * n, "table_bytes": ctx.table_bytes,
                   "l2": "inputs (raw events) are larger than L2; no flush needed",
                   "jobs": "one independent job of this size per GPU"},
        "raw_event_gbs": 32 * value / 1e9,
        "hbm_frac_step": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
        "hbm_frac_step_vs_8tbs": step_bytes / (ms_step * 1e-3) / 1e9 / 8000.0,
        "roofline": {"bound": "hbm", "kernel": "aggregate_seg_kernel" if not s.shuffle else
                     "argus_aggregate = partition_count/offsets/scan/scatter + aggregate_seg_kernel",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "peak_source": peak_src, "kernel_ms": agg_ms,
                     "algorithmic_bytes": alg_bytes, "share_of_step": agg_ms / ms_step},
        "clocks": clocks, "e2e": e2e, "gpu_launches": (8 if s.shuffle else 4) * args.steps,
        "counters": {"n_valid": n_valid, "n_invalid": n_invalid},
    }
    if world.size == 1 and not args.no_cpu_baseline:
        sample_ranks = max(1, min(s.n_ranks, (160_000_000 // (s.n_steps * s.n_events)) or 1))
        n_ev, dt = oracle_sample(wl, sample_ranks, os.cpu_count() or 1)
        out["cpu_baseline"] = {"value": n_ev / dt, "unit": "events/s", "cores": 1, "kind": "oracle",
                               "sample": f"first {sample_ranks} of {s.n_ranks} ranks ({n_ev} events) of "
                                         f"'{s.name}', aggregate + phase_times + diagnose, {dt:.1f} s; "
                                         f"host has {os.cpu_count()} cores (generator used them, oracle 1)"}
    print(json.dumps(out))
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="production",
                    help="tiny | mid | scale | unsorted | production (BASELINE.json configs[0..4])")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", type=int, default=0, help="segmented-kernel geometry (tuning)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    from paper_2606_20374_b200 import dist as D
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        if rank == 0:
            run_reference(args, D.World())
        return
    world = D.init_world(args.gpus)
    try:
        run_ours(args, world)
    finally:
        D.finish(world)


if __name__ == "__main__":
    main()
