#!/usr/bin/env python
"""bench.py — the ARGUS hot path on B200: raw kernel events -> per-(rank, step, sig) summaries and
spans -> cross-rank median/MAD diagnosis (BASELINE.json `metric`), on seeded synthetic events.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload production] [--impl ours|reference]
                  [--scaling weak|strong] [--exchange a2a|p2p] [--bimodal F] [--no-e2e] [--no-cpu-baseline] [--no-next]

One step = one pass of the whole path over the workload: argus_reset + argus_aggregate +
argus_phase_times + argus_diagnose.  `value` is timed with CUDA events with the events resident in
HBM; `e2e` is the same step through argus_aggregate_host with HOST (pinned) buffers: the 256 MiB
chunked host->device copies and the device->host read of the diagnosis are inside the timed region,
and its outputs are compared with the resident leg's.  `next_rows` times every NEXT-row call (KDE
clustering, record encodings, L3 / L2 / L1) alone on the finalised table, outside the step.  Prints ONE
JSON line on rank 0.
`--impl reference` times the CPU oracle (oracle/) instead.  `--gpus N` (N > 1) outside torchrun
re-launches itself under torch.distributed.run with N ranks, or fails if the box has fewer GPUs.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
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
        self.ready = threading.Event()       # the first sample has been taken
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
                self.ready.set()
                time.sleep(0.002)
        except Exception as e:  # NVML missing: report it, do not fail the bench
            self.err = repr(e)
            self.ready.set()

    def begin(self):
        """Start sampling; returns once the first sample is in (short timed regions still get clocks)."""
        self.start()
        self.ready.wait(timeout=5)
        self.samples.clear()
        return self

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
    """Time the oracle, as it stands (one thread), on the first `n_ranks_sample` ranks of the
    workload; the events are expanded on the host in blocks of ranks (untimed) so that a whole config
    fits host memory.  Returns (events, oracle seconds, oracle object)."""
    from oracle import Oracle
    s = wl.spec
    dt, n_ev = 0.0, 0
    if s.shuffle:
        ev = wl.expand_host(0, s.n_ranks, threads=threads)
        ev = ev[: n_ranks_sample * s.n_steps * s.n_events]
        o = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
        t0 = time.perf_counter()
        o.aggregate(ev)
        dt += time.perf_counter() - t0
        n_ev = ev.size
    else:
        o = Oracle(n_ranks_sample, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
        block = max(1, 40_000_000 // (s.n_steps * s.n_events))       # ~1.3 GB of events per block
        for lo in range(0, n_ranks_sample, block):
            ev = wl.expand_host(lo, min(n_ranks_sample, lo + block), threads=threads)
            t0 = time.perf_counter()
            o.aggregate(ev)
            dt += time.perf_counter() - t0
            n_ev += ev.size
    t0 = time.perf_counter()
    o.phase_times()
    o.diagnose()
    dt += time.perf_counter() - t0
    return n_ev, dt, o


def workload_config(s):
    """The `config` object of the JSON line: the workload and what the timing rules ask to be said about it.
    The same keys and values on both arms (the driver compares them)."""
    n = s.total_events
    return {"workload": s.name, "n_ranks": s.n_ranks, "n_steps": s.n_steps,
            "events_per_rank_step": s.n_events, "n_sigs": s.n_sigs, "n_phases": s.n_phases,
            "events": n, "raw_bytes": 32 * n,
            "table_bytes": s.n_ranks * s.n_steps * (64 + 32 * (s.n_phases + 1) + 160 * s.n_sigs),
            "l2": "inputs (raw events) are larger than L2; no flush needed",
            "jobs": "one independent job of this size per GPU"}


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
        n_ev, dt, _ = oracle_sample(wl, sample_ranks, threads)
        if i >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    v = n_ev / t
    sample = f"first {sample_ranks} of {s.n_ranks} ranks ({n_ev} events) of '{s.name}' per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": workload_config(s),
        "raw_event_gbs": 32 * v / 1e9,
        "cpu_baseline": {"value": v, "unit": "events/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ---------------------------------------------------------------------------------------------
def _ms(pairs):
    return [a.elapsed_time(b) for a, b in pairs]


def next_rows(ctx, rec, d_ev, s, peak, reps=5, l3_keys=4096, fine_limit_bytes=24 << 30):
    """The SURVEY 8(f) NEXT rows on the table the timed steps left behind (finalised), each call timed alone
    with CUDA events (1 warm-up, median of `reps`); outside the step's timed region.  Bytes are the
    algorithmic ones of DESIGN.md 6.6 / 6.7 (what the call must read and write), GB/s = bytes / median time.
    Nothing here is compared with the oracle (tests/test_paper_literal_gpu.py, tests/test_compact_gpu.py do)."""
    import torch
    R, T, S, P = s.n_ranks, s.n_steps, s.n_sigs, s.n_phases
    n, n_cells, K, MC = s.total_events, R * T * S, T * S, 8
    dev = rec.device
    mk = lambda: torch.cuda.Event(enable_timing=True)

    def timed(fn, reset=None):
        ts = []
        for i in range(reps + 1):
            if reset is not None:
                reset()
            a, b = mk(), mk()
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            if i:
                ts.append(a.elapsed_time(b))
        return float(np.median(ts)), float(np.min(ts))

    def line(ms, best, nbytes, bound, **kw):
        d = {"ms": ms, "ms_best": best, "algorithmic_bytes": int(nbytes), "gbs": nbytes / (ms * 1e-3) / 1e9,
             "hbm_frac": nbytes / (ms * 1e-3) / 1e9 / peak, "bound": bound}
        d.update(kw)
        return d

    out = {}
    u8 = lambda m: torch.zeros(m, dtype=torch.uint8, device=dev)
    # NEXT-1 on the records' own 32-bucket histograms: read 128 B of histogram per cell, write MC triples + 1 B
    d_c, d_n = u8(n_cells * MC * 8), u8(n_cells)
    p32 = ctx.kde_params(per_octave=1, n_bins=32, max_clusters=MC)
    ms, best = timed(lambda: ctx.kde_clusters_records(rec, p32, d_c, d_n))
    ncl = d_n.to(torch.int64)
    n_clusters = int(ncl.sum())
    out["next1_kde_records"] = line(ms, best, n_cells * (128 + 8 * MC + 1), "hbm (a thread per narrow cell; fp64 exp only for cells that can hold a valley)",
                                    cells=n_cells, cells_per_s=n_cells / (ms * 1e-3), clusters=n_clusters,
                                    cells_with_2plus=int((ncl >= 2).sum()))
    # NEXT-4b record encodings: read the table once, write the stream
    tb = ctx.table_bytes
    off = torch.zeros(R * T + 1, dtype=torch.int64, device=dev)
    buf = u8(ctx.sparse_bound())
    ms, best = timed(lambda: ctx.sparse_encode(rec, buf, off))
    sparse_len = int(off[-1])
    out["next4_sparse_encode"] = line(ms, best, tb + sparse_len, "hbm", stream_bytes=sparse_len,
                                      raw_over_record=32 * n / sparse_len, dense_over_record=tb / sparse_len,
                                      bytes_per_rank_step=sparse_len / (R * T))
    del buf
    buf = u8(ctx.triple_bound(MC))
    ms, best = timed(lambda: ctx.triple_encode(rec, d_c, d_n, MC, buf, off))
    triple_len = int(off[-1])
    out["next4_triple_encode"] = line(ms, best, R * T * (64 + 32 * (P + 1)) + n_cells * (8 * MC + 1) + triple_len, "hbm",
                                      stream_bytes=triple_len, raw_over_record=32 * n / triple_len,
                                      bytes_per_rank_step=triple_len / (R * T), triples_per_rank_step=n_clusters / (R * T),
                                      paper="~3,700x: ~10 MB -> ~2.7 KB, ~200 triples per rank per step (PAPER.md:196; "
                                            "its key is (kernel, stream, rank) with a few hundred kernels, this workload "
                                            "has S sigs per rank-step)")
    del buf
    # NEXT-1 on the fine grid (8 bins per octave): events -> [R][T][S][256] u32 with L2 atomics -> clusters
    fine_bytes = n_cells * 1024
    if d_ev is not None and fine_bytes <= fine_limit_bytes:
        hist = torch.zeros(n_cells * 256, dtype=torch.int32, device=dev)
        ms, best = timed(lambda: ctx.fine_hist(d_ev, n, hist), reset=lambda: hist.zero_())
        out["next1_fine_hist"] = line(ms, best, 32 * n + fine_bytes, "hbm + L2 atomics", events_per_s=n / (ms * 1e-3))
        d_c8, d_n8 = u8(n_cells * MC * 8), u8(n_cells)
        p256 = ctx.kde_params(max_clusters=MC)
        ms, best = timed(lambda: ctx.kde_clusters(hist, n_cells, p256, d_c8, d_n8))
        out["next1_kde_fine"] = line(ms, best, n_cells * (1024 + 8 * MC + 1), "hbm (1 KB of counters per cell) / alu",
                                     cells=n_cells, cells_per_s=n_cells / (ms * 1e-3), clusters=int(d_n8.sum()))
        del hist, d_n8
    else:
        d_c8 = None
        out["next1_fine_hist"] = {"skipped": f"[R][T][S][256] u32 = {fine_bytes / 2**30:.1f} GiB: measured on mid / scale"}
    # NEXT-2: regroup the triples per key, then score the first l3_keys keys over all R ranks
    d_cnt = torch.zeros(K * R * MC, dtype=torch.int32, device=dev)
    d_p50 = torch.zeros(K * R * MC, dtype=torch.float64, device=dev)
    d_p99 = torch.zeros(K * R * MC, dtype=torch.float64, device=dev)
    ms, best = timed(lambda: ctx.clusters_to_l3(d_c, MC, 1, d_cnt, d_p50, d_p99))
    out["next2_clusters_to_l3"] = line(ms, best, n_cells * MC * (8 + 20), "hbm (transpose)")
    kk = min(K, l3_keys)
    G = 256
    d_score = torch.zeros(kk * R, dtype=torch.float64, device=dev)
    d_stat = torch.zeros(kk * 5, dtype=torch.float64, device=dev)
    d_fl = u8(kk * R)
    def l3_row(n_keys, what):
        c0 = ctx.l3_path_count()
        ms, best = timed(lambda: ctx.l3_detect(d_cnt, d_p50, d_p99, n_keys, R, MC, d_score, d_stat, d_fl, n_grid=G))
        c1 = ctx.l3_path_count()
        per = [(b - a) // (reps + 1) for a, b in zip(c0, c1)]            # counted by the kernel, per call
        bound = "alu / shared memory: " + ("class path (weighted sums over <= 256 classes of identical mixtures)"
                                           if per[1] == 0 else
                                           "general path (a sort of R CDF values per grid point)" if per[0] == 0 else
                                           "class path and general path mixed, see keys_*") + "; " + what
        return line(ms, best, n_keys * R * (MC * 20 + 9), bound, keys=n_keys, ranks=R, n_grid=G,
                    keys_class_path=per[0], keys_general_path=per[1], keys_empty=per[2], us_per_key=ms * 1e3 / n_keys,
                    cdf_points_per_s=n_keys * R * G / (ms * 1e-3), flagged=int(d_fl[:n_keys * R].sum()))
    out["next2_l3_detect"] = l3_row(kk, "clusters of the records' 32-bucket histograms")
    if d_c8 is not None:
        # NEXT-2 on the clusters of the FINE grid (8 bins per octave, what PAPER.md:178 describes): ranks rarely share
        # a mixture there, so this is the general path of the L3 kernel (a sort of R CDF values per grid point)
        kf = min(K, 512)
        ctx.clusters_to_l3(d_c8, MC, 8, d_cnt, d_p50, d_p99)
        out["next2_l3_detect_fine"] = l3_row(kf, "clusters of the fine grid (8 bins per octave)")
        del d_c8
    del d_cnt, d_p50, d_p99, d_c, d_n
    # NEXT-3: L2 over every phase span (one group per 8 consecutive ranks), L1 over the R iteration-time series
    route = u8(P + 1)
    gid = (torch.arange(R, device=dev, dtype=torch.int32) // 8 * 8).contiguous()
    d_groups = u8((P + 1) * R * 32)
    d_z = torch.zeros((P + 1) * R, dtype=torch.float64, device=dev)
    d_xb = torch.zeros((P + 1) * R, dtype=torch.float64, device=dev)
    d_f2 = u8((P + 1) * R)
    ms, best = timed(lambda: ctx.l2_groups(rec, route, gid, 3.0, d_groups, d_z, d_f2, d_xb))
    out["next3_l2_groups"] = line(ms, best, R * T * (P + 1) * 32 + (P + 1) * R * (32 + 8 + 1), "latency (KBs of data)")
    if 8 <= T <= 2048:
        spans = torch.zeros(R * T * (P + 1) * 32, dtype=torch.uint8, device=dev)
        ctx.phase_times(rec, spans)
        d_l1 = u8(R * 216)
        ms, best = timed(lambda: ctx.l1_detect(spans.data_ptr() + P * 32 + 16, T * (P + 1) * 32, (P + 1) * 32, R, T, d_l1))
        out["next3_l1_detect"] = line(ms, best, R * T * 8 + R * 216, "latency (KBs of data)")
    return out


def run_ours(args, world):
    import torch
    from paper_2606_20374_b200 import argus as A
    from paper_2606_20374_b200 import dist as D
    from paper_2606_20374_b200.workload import build_workload
    import dataclasses

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    if args.scaling == "strong":
        from paper_2606_20374_b200 import sharded
        return sharded.bench_strong(args, world, METRIC, measured_peak_gbs, ClockSampler)
    torch.cuda.set_device(world.local_rank)
    dev = world.local_rank
    wl0 = build_workload(args.workload)
    if args.bimodal > 0.0:
        wl0 = build_workload(dataclasses.replace(wl0.spec, bimodal_frac=args.bimodal,
                                                 name=wl0.spec.name + f"+bimodal{args.bimodal:g}"))
    if args.sigs > 0:
        # the paper's key count (~100 active (kernel, stream) combinations, ~2 clusters each) on the
        # named workload's event volume: the like-for-like figure beside "~10 MB -> ~2.7 KB" (context, not a target)
        wl0 = build_workload(dataclasses.replace(wl0.spec, n_sigs=args.sigs, name=wl0.spec.name + f"+sigs{args.sigs}"))
    spec = dataclasses.replace(wl0.spec, seed=D.job_seed(wl0.spec.seed, world))
    wl = build_workload(spec) if world.rank else wl0
    s = wl.spec
    n = s.total_events

    d_ev = wl.expand_device(device=f"cuda:{dev}")
    ctx = A.Argus(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base, sorted_hint=not s.shuffle,
                  device=dev, max_ungrouped_events=n if s.shuffle else 0,
                  max_spill_events=min(n // 4, 2**32 - 1) if args.spill < 0 else args.spill)
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
        if ev_pairs is not None:
            ev_pairs[2].record()

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    D.barrier(world)

    sampler = ClockSampler(dev).begin()
    mk = lambda: torch.cuda.Event(enable_timing=True)
    t_beg, t_end = mk(), mk()
    marks = [(mk(), mk(), mk()) for _ in range(args.steps)]
    k0, m0 = ctx.launch_count()
    torch.cuda.synchronize()
    t_beg.record()
    for i in range(args.steps):
        step(marks[i])
    t_end.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    k1, m1 = ctx.launch_count()
    D.barrier(world)
    ms_total = D.max_over_ranks(world, t_beg.elapsed_time(t_end))
    ms_step = ms_total / args.steps
    agg_list = _ms([(a, b) for a, b, _ in marks])
    agg_ms = float(np.mean(agg_list))
    # per-step durations (reset of step i+1 is two tiny memsets: attributed to the step they precede)
    step_list = [marks[i][0].elapsed_time(marks[i][2]) for i in range(args.steps)]
    n_valid, n_invalid = ctx.stats()
    n_requeued, n_overflow = ctx.refused_count()
    total_events = D.sum_over_ranks(world, float(n))
    value = total_events / (ms_step * 1e-3)
    resident = {k: v.clone() for k, v in outs.items()}

    # ---- the NEXT rows of SURVEY 8(f) on the finalised table (outside the timed steps) --------------
    nxt = None
    if world.rank == 0 and not args.no_next:
        try:
            nxt = next_rows(ctx, rec, d_ev, s, measured_peak_gbs()[0])
        except Exception as e:
            nxt = {"error": repr(e)[:300]}
        torch.cuda.synchronize()

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
            rec_keep = rec.clone()
            # The summary leaves the device too (NS (5): the reducer uploads the compressed
            # records): the paper's (count, p50, p99) TRIPLE stream of every rank-step, encoded after the
            # diagnosis and copied to pinned host memory with its offsets, all inside the timed region.
            MC = 8
            n_cells = s.n_ranks * s.n_steps * s.n_sigs
            n_rec = s.n_ranks * s.n_steps
            p32 = ctx.kde_params(per_octave=1, n_bins=32, max_clusters=MC)
            d_c = torch.zeros(n_cells * MC * 8, dtype=torch.uint8, device=f"cuda:{dev}")
            d_n = torch.zeros(n_cells, dtype=torch.uint8, device=f"cuda:{dev}")
            d_stream = torch.empty(ctx.triple_bound(MC), dtype=torch.uint8, device=f"cuda:{dev}")
            d_off = torch.zeros(n_rec + 1, dtype=torch.int64, device=f"cuda:{dev}")
            ctx.kde_clusters_records(rec, p32, d_c, d_n)          # the resident leg's stream (rec is finalised)
            ctx.triple_encode(rec, d_c, d_n, MC, d_stream, d_off)
            ref_len = int(d_off[-1])
            ref_stream, ref_off = d_stream[:ref_len].cpu(), d_off.cpu()
            h_stream = torch.empty(d_stream.numel(), dtype=torch.uint8, pin_memory=True)
            h_off = torch.empty(n_rec + 1, dtype=torch.int64, pin_memory=True)
            h_len = torch.zeros(1, dtype=torch.int64, pin_memory=True)
            d_stream.zero_(); d_off.zero_()
            for v in outs.values():
                v.zero_()
            shipped = [0]

            def e2e_step():
                ctx.reset(rec)
                ctx.aggregate_host(h_ev, n, chunk, d_ring, RING_SLOTS, rec)
                ctx.phase_times(rec)
                ctx.diagnose(rec, outs)
                ctx.kde_clusters_records(rec, p32, d_c, d_n)
                ctx.triple_encode(rec, d_c, d_n, MC, d_stream, d_off)
                for k in outs:
                    h_out[k].copy_(outs[k], non_blocking=True)
                h_off.copy_(d_off, non_blocking=True)
                h_len.copy_(d_off[-1:], non_blocking=True)
                torch.cuda.current_stream().synchronize()     # the stream's length is known only now (8 bytes)
                shipped[0] = int(h_len[0])
                h_stream[:shipped[0]].copy_(d_stream[:shipped[0]], non_blocking=True)

            e2e_steps = max(1, min(args.steps, args.e2e_steps))
            e2e_step()
            torch.cuda.synchronize()
            D.barrier(world)
            a, b = mk(), mk()
            a.record()
            for _ in range(e2e_steps):
                e2e_step()
            b.record()
            torch.cuda.synchronize()
            e_ms = D.max_over_ranks(world, a.elapsed_time(b)) / e2e_steps
            # the e2e leg checks itself: same table bytes, same six outputs (device and host copies),
            # same counters as the resident leg
            nv2, ni2 = ctx.stats()
            verified = bool(torch.equal(rec, rec_keep)) and (nv2, ni2) == (n_valid, n_invalid)
            for k in outs:
                verified = verified and bool(torch.equal(outs[k], resident[k])) and \
                    bool(torch.equal(h_out[k], resident[k].cpu()))
            # ... and the shipped record stream, byte for byte, with the one encoded from the resident leg's table
            verified = verified and shipped[0] == ref_len and bool(torch.equal(h_off, ref_off)) and \
                bool(torch.equal(h_stream[:ref_len], ref_stream))
            d2h += ref_len + h_off.numel() * 8 + 8
            del rec_keep, d_c, d_n, d_stream, ref_stream
            # overlap efficiency max(t_copy, t_agg) / t_total: the copies alone through
            # the same ring on the copy stream (argus_ingest), the aggregation alone from the resident
            # leg, and the overlapped host-streamed aggregation
            cs = torch.cuda.Stream()
            with torch.cuda.stream(cs):
                c0, c1 = mk(), mk()
                c0.record()
                for c, lo in enumerate(range(0, n, chunk)):
                    cnt = min(chunk, n - lo)
                    ctx.ingest(h_ev.data_ptr() + lo * 32, cnt, d_ring.data_ptr() + (c % RING_SLOTS) * chunk * 32, cs)
                c1.record()
            torch.cuda.synchronize()
            t_copy = c0.elapsed_time(c1)
            g0, g1 = mk(), mk()
            ctx.reset(rec)
            g0.record()
            ctx.aggregate_host(h_ev, n, chunk, d_ring, RING_SLOTS, rec)
            g1.record()
            torch.cuda.synchronize()
            t_total = g0.elapsed_time(g1)
            ctx.phase_times(rec)                  # leave a finalised table behind (parity_check below)
            torch.cuda.synchronize()
            e2e = {"value": total_events / (e_ms * 1e-3), "unit": "events/s", "ms_per_step": e_ms,
                   "steps": e2e_steps, "h2d_bytes_per_step": 32 * n, "d2h_bytes_per_step": d2h,
                   "h2d_gbs": 32 * n / (e_ms * 1e-3) / 1e9, "chunk_bytes": chunk * 32,
                   "ring_slots": RING_SLOTS, "verified": verified,
                   "shipped": {"encoding": "triple (R38: per cell its (count, p50, p99) clusters, max 8) + offsets + "
                                           "the six diagnosis outputs", "stream_bytes": ref_len,
                               "raw_over_stream": 32 * n / max(1, ref_len)},
                   "overlap": {"t_copy_ms": t_copy, "t_agg_ms": agg_ms, "t_total_ms": t_total,
                               "efficiency": max(t_copy, agg_ms) / t_total}}
        except Exception as e:  # e.g. the box cannot pin the whole buffer
            e2e = {"value": None, "unit": "events/s", "error": repr(e)[:200],
                   "h2d_bytes_per_step": 32 * n, "d2h_bytes_per_step": None}

    # ---- N > 1: the SAME workload once more as ONE job sharded by trace rank: aggregation per
    # shard, one exchange of the 8-byte-per-cell sum plane, selection per sig slice.  Reported beside the
    # weak-scaling headline, never instead of it; unmeasured on hardware so far, hence guarded.
    sharded_job = None
    if world.size > 1 and args.scaling == "both" and not s.shuffle and args.bimodal == 0.0 and args.sigs == 0:
        try:
            from paper_2606_20374_b200 import sharded
            torch.cuda.empty_cache()
            sharded_job = sharded.bench_strong(args, world, METRIC, measured_peak_gbs, ClockSampler, emit=False)
        except Exception as e:
            sharded_job = {"error": repr(e)[:300]}

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
        "warmup": args.warmup, "ms_per_step": ms_step, "ms_per_step_median": float(np.median(step_list)),
        "ms_per_step_best": float(np.min(step_list)), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": workload_config(s), "workspace_bytes": ctx.workspace_bytes,
        "raw_event_gbs": 32 * value / 1e9,
        "hbm_frac_step": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
        "hbm_frac_step_vs_8tbs": step_bytes / (ms_step * 1e-3) / 1e9 / 8000.0,
        "roofline": {"bound": "hbm", "kernel": "aggregate_seg_kernel" if not s.shuffle else
                     "argus_aggregate = grouping pass + aggregate_seg_kernel",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic,
                     "traffic_source": None if traffic is None else
                     f"committed ncu --set full capture profiles/{s.name}_seg_traffic.txt (a constant read from that "
                     "file, not measured in this run)", "peak_source": peak_src, "kernel_ms": agg_ms,
                     "kernel_ms_median": float(np.median(agg_list)), "kernel_ms_best": float(np.min(agg_list)),
                     "algorithmic_bytes": alg_bytes, "share_of_step": agg_ms / ms_step},
        "clocks": clocks, "e2e": e2e,
        "gpu_launches": k1 - k0, "gpu_memsets": m1 - m0,     # counted by the library (argus_launch_count)
        # events a compact shared-memory cell refused (range wider than four log2 buckets, >= 2^32 ns), per step:
        # re-queued through the spill area and replayed at the flush of their rank-step / taken one by one by L2 reductions
        "counters": {"n_valid": n_valid, "n_invalid": n_invalid, "n_requeued": n_requeued,
                     "n_overflow": n_overflow, "requeued_frac": n_requeued / max(1, n_valid),
                     "overflow_frac": n_overflow / max(1, n_valid)},
    }
    if args.bimodal > 0.0:
        out["config"]["bimodal_sigs"] = wl.n_bimodal
    if nxt is not None:
        out["next_rows"] = nxt
    if sharded_job is not None:
        out["sharded_job"] = sharded_job
    if world.size == 1 and not args.no_cpu_baseline:
        k = args.cpu_baseline_ranks if args.cpu_baseline_ranks > 0 else s.n_ranks
        if args.cpu_baseline_ranks < 0:      # default: a bounded sample, about 15 s of oracle time
            k = max(1, min(s.n_ranks, (670_000_000 // (s.n_steps * s.n_events)) or 1))
        if s.shuffle:
            k = s.n_ranks
        n_ev, dt, o = oracle_sample(wl, k, os.cpu_count() or 1)
        out["cpu_baseline"] = {"value": n_ev / dt, "unit": "events/s", "cores": 1, "kind": "oracle",
                               "sample": f"first {k} of {s.n_ranks} ranks ({n_ev} events) of "
                                         f"'{s.name}', aggregate + phase_times + diagnose, {dt:.1f} s; "
                                         f"host has {os.cpu_count()} cores (generator used them, oracle 1)"}
        # bit-exact check of this very run: the table rows of the sampled ranks (every byte of their
        # records; the e2e leg above left the same table, see e2e.verified) against the oracle's
        want = o.records()
        rb = ctx.record_bytes
        got = rec[: want.shape[0] * rb].cpu().numpy().reshape(want.shape)
        out["parity_check"] = {"ranks": int(k), "records_equal_oracle": bool(np.array_equal(got, want)),
                               "counters_equal_oracle": (n_valid, n_invalid) == (o.n_valid, o.n_invalid)
                               if k == s.n_ranks else None}
    print(json.dumps(out))
    ctx.close()


def relaunch_under_torchrun(args) -> int:
    """`python bench.py --gpus N` outside torchrun: spawn N ranks (one per GPU) or fail loudly."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        print(f"bench.py: --gpus {args.gpus} but this box has {have} CUDA device(s)", file=sys.stderr)
        return 2
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="production",
                    help="tiny | mid | scale | unsorted | production (BASELINE.json configs[0..4])")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default=None, choices=["weak", "strong", "both"],
                    help="N > 1: weak = one job of the named size per GPU; strong = ONE job sharded by trace rank; "
                         "both (the default for N > 1) = the weak line with the sharded job's numbers under "
                         "\"sharded_job\"; N = 1 defaults to weak")
    ap.add_argument("--exchange", default="a2a", choices=["a2a", "p2p"],
                    help="--scaling strong: all_to_all_single (NCCL) or peer stores through symmetric memory")
    ap.add_argument("--bimodal", type=float, default=0.0,
                    help="stress knob: share of the sigs with a second duration mode 8-64x the first (PAPER.md:166)")
    ap.add_argument("--sigs", type=int, default=0,
                    help="override the workload's signature count (e.g. 128: the paper's ~100 keys per rank)")
    ap.add_argument("--spill", type=int, default=-1,
                    help="argus_config.max_spill_events: -1 = a quarter of the events (default), 0 = no spill area")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next", action="store_true",
                    help="skip the separately timed NEXT rows (KDE clusters, record encodings, L3 / L2 / L1)")
    ap.add_argument("--cpu-baseline-ranks", type=int, default=-1,
                    help="ranks of the workload the oracle is timed on: -1 = bounded sample (default), 0 = all")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.scaling is None:
        args.scaling = "both" if args.gpus > 1 else "weak"
    from paper_2606_20374_b200 import dist as D
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        if rank == 0:
            run_reference(args, D.World())
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args))
    world = D.init_world(args.gpus)
    try:
        run_ours(args, world)
    finally:
        D.finish(world)


if __name__ == "__main__":
    main()
