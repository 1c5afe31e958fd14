"""ONE job sharded by trace rank over G GPUs (the paper's comparison of
"the same kernel across different ranks", when the ranks' events live on different
devices).  Host-side plumbing only: which ranks and sigs a GPU owns, the send/receive layouts of the
one exchange, and the calls into the C ABI (argus_pack_planes / argus_diagnose_planes).  Every number
is produced by the kernels behind the ABI.

Data flow on GPU g of G (contiguous balanced splits):

  aggregate + phase_times      its ranks [r0_g, r0_g + R_g), ctx of n_ranks = R_g       no exchange
  pack                         for every destination d: its ranks' sums of d's sig slice [s0_d, s1_d),
                               rank-contiguous, [T][S_d][R_g]; and its span plane [T][P+1][R_g]
  exchange                     "a2a": one all_to_all_single of the sig planes (8 B per cell of the job in
                               total: 134 MB at production, 16.8 MB per GPU on 8) + one all_gather of
                               the span planes (a few KB), torch.distributed (NCCL over NVLink/NVSwitch);
                               "p2p": the pack kernel stores straight into the owner's [T][S_d][R] plane
                               through peer-mapped pointers (torch symmetric memory), rows of R_g
                               contiguous u64, then one barrier
  diagnose_planes              sig series of its slice over ALL R ranks; span series (tiny) replicated
  roll-up                      rank_score partials summed with one all_reduce
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence, Tuple

import numpy as np
import torch


def split(n: int, parts: int) -> List[Tuple[int, int]]:
    """Contiguous balanced split of range(n): the first n % parts shares get one more."""
    q, r = divmod(n, parts)
    out, lo = [], 0
    for i in range(parts):
        hi = lo + q + (1 if i < r else 0)
        out.append((lo, hi))
        lo = hi
    return out


@dataclasses.dataclass
class Layout:
    """Who owns what in a job of R ranks, T steps, S sigs, P phases over G GPUs."""
    G: int
    R: int
    T: int
    S: int
    P: int

    @property
    def ranks(self):
        return split(self.R, self.G)

    @property
    def sigs(self):
        return split(self.S, self.G)

    def send_counts(self, g: int) -> List[int]:
        """u64 elements GPU g sends to each destination d: T * S_d * R_g."""
        rg = self.ranks[g][1] - self.ranks[g][0]
        return [self.T * (s1 - s0) * rg for s0, s1 in self.sigs]

    def recv_counts(self, d: int) -> List[int]:
        """u64 elements GPU d receives from each source g: T * S_d * R_g."""
        sd = self.sigs[d][1] - self.sigs[d][0]
        return [self.T * sd * (r1 - r0) for r0, r1 in self.ranks]


def assemble_sig_plane(lay: Layout, d: int, recv: torch.Tensor, out: Optional[torch.Tensor] = None):
    """recv: what GPU d got from the all-to-all, sources concatenated, source g's part laid out
    [T][S_d][R_g].  Returns the plane [T][S_d][R] (rank-contiguous over ALL ranks).  Data movement only."""
    s0, s1 = lay.sigs[d]
    sd = s1 - s0
    if out is None:
        out = torch.empty(lay.T * sd * lay.R, dtype=recv.dtype, device=recv.device)
    plane = out.view(lay.T * sd, lay.R)
    off = 0
    for (r0, r1), cnt in zip(lay.ranks, lay.recv_counts(d)):
        plane[:, r0:r1] = recv[off:off + cnt].view(lay.T * sd, r1 - r0)
        off += cnt
    return out


def assemble_span_plane(lay: Layout, parts: Sequence[torch.Tensor], out: Optional[torch.Tensor] = None):
    """parts[g]: GPU g's span plane [T][P+1][R_g].  Returns [T][P+1][R]."""
    rows = lay.T * (lay.P + 1)
    if out is None:
        out = torch.empty(rows * lay.R, dtype=parts[0].dtype, device=parts[0].device)
    plane = out.view(rows, lay.R)
    for (r0, r1), p in zip(lay.ranks, parts):
        plane[:, r0:r1] = p.view(rows, r1 - r0)
    return out


class Shard:
    """GPU g's part of the job: its ctx (n_ranks = R_g), table, send buffers and slice outputs."""

    def __init__(self, lay: Layout, g: int, step_base: int = 0, device: int = 0, sorted_hint: bool = True,
                 max_ungrouped_events: int = 0):
        from . import argus as A
        self.lay, self.g, self.device = lay, g, device
        self.r0, self.r1 = lay.ranks[g]
        self.s0, self.s1 = lay.sigs[g]
        self.ctx = A.Argus(self.r1 - self.r0, lay.T, lay.S, lay.P, step_base, sorted_hint=sorted_hint,
                           device=device, max_ungrouped_events=max_ungrouped_events)
        dev = f"cuda:{device}"
        self.rec = self.ctx.alloc_records()
        self.send = torch.empty(sum(lay.send_counts(g)), dtype=torch.int64, device=dev)
        self.span_part = torch.empty(lay.T * (lay.P + 1) * (self.r1 - self.r0), dtype=torch.int64, device=dev)
        sd, T, R, P = self.s1 - self.s0, lay.T, lay.R, lay.P
        u8 = torch.uint8
        self.outs = dict(sig_stats=torch.empty(T * sd * 32, dtype=u8, device=dev),
                         sig_flags=torch.empty(T * sd * R, dtype=u8, device=dev),
                         span_stats=torch.empty(T * (P + 1) * 32, dtype=u8, device=dev),
                         span_flags=torch.empty(T * (P + 1) * R, dtype=u8, device=dev),
                         rank_score=torch.empty(T * R, dtype=torch.int32, device=dev),
                         step_anomalous=torch.empty(T, dtype=torch.int32, device=dev))

    # ---- phases (each a few calls into the C ABI) -------------------------------------------------
    def aggregate(self, d_events, n: int, stream=None) -> None:
        """Events of this shard's ranks, rank field RELATIVE to r0 (rank - r0)."""
        self.ctx.reset(self.rec, stream)
        self.ctx.aggregate(d_events, n, self.rec, stream)
        self.ctx.phase_times(self.rec, None, stream)

    def pack_for_all_to_all(self, stream=None) -> None:
        """send = for d in 0..G-1: [T][S_d][R_g]; span_part = [T][P+1][R_g]."""
        rg = self.r1 - self.r0
        off = 0
        for d, ((s0, s1), cnt) in enumerate(zip(self.lay.sigs, self.lay.send_counts(self.g))):
            self.ctx.pack_planes(self.rec, s0, s1, self.send.data_ptr() + off * 8 if cnt else None,
                                 self.span_part if d == 0 else None, rg, 0, stream)
            off += cnt

    def pack_into_planes(self, sig_plane_ptrs: Sequence[int], span_plane_ptrs: Sequence[int], stream=None) -> None:
        """p2p: store this shard's columns straight into every owner's [T][S_d][R] plane (peer-mapped
        or local pointers) and into every GPU's span plane."""
        for d, (s0, s1) in enumerate(self.lay.sigs):
            self.ctx.pack_planes(self.rec, s0, s1, sig_plane_ptrs[d] if s1 > s0 else None, span_plane_ptrs[d],
                                 self.lay.R, self.r0, stream)

    def diagnose(self, sig_plane, span_plane, stream=None) -> None:
        self.ctx.diagnose_planes(sig_plane if self.s1 > self.s0 else None, span_plane, self.lay.R, self.lay.R,
                                 self.s1 - self.s0, self.outs, stream)

    def outs_to_host(self) -> dict:
        from . import argus as A
        lay, sd = self.lay, self.s1 - self.s0
        o = self.outs
        return dict(sig_stats=o["sig_stats"].cpu().numpy().view(A.STAT_DTYPE).reshape(lay.T, sd),
                    sig_flags=o["sig_flags"].cpu().numpy().reshape(lay.T, sd, lay.R),
                    span_stats=o["span_stats"].cpu().numpy().view(A.STAT_DTYPE).reshape(lay.T, lay.P + 1),
                    span_flags=o["span_flags"].cpu().numpy().reshape(lay.T, lay.P + 1, lay.R),
                    rank_score=o["rank_score"].cpu().numpy().view(np.uint32).reshape(lay.T, lay.R),
                    step_anomalous=o["step_anomalous"].cpu().numpy().view(np.uint32).reshape(lay.T))

    def close(self) -> None:
        self.ctx.close()


def merge_outputs(lay: Layout, per_shard: Sequence[dict]) -> dict:
    """Whole-job outputs from the shards' slice outputs (host side, for tests and reports): sig series
    concatenated along the sig axis, rank_score partials summed, span outputs taken from shard 0."""
    return dict(sig_stats=np.concatenate([o["sig_stats"] for o in per_shard], axis=1),
                sig_flags=np.concatenate([o["sig_flags"] for o in per_shard], axis=1),
                span_stats=per_shard[0]["span_stats"], span_flags=per_shard[0]["span_flags"],
                rank_score=np.sum([o["rank_score"] for o in per_shard], axis=0, dtype=np.uint32),
                step_anomalous=per_shard[0]["step_anomalous"])


# ---- the exchange over torch.distributed (one process per GPU) ----------------------------------------
def exchange_all_to_all(lay: Layout, g: int, send: torch.Tensor, span_part: torch.Tensor, group=None):
    """One all_to_all_single (sig planes) + one all_gather (span planes).  Works on NCCL (device
    tensors) and gloo (CPU tensors: the world-of-two test).  Returns (sig plane [T][S_g][R], span
    plane [T][P+1][R]) of GPU g."""
    import torch.distributed as dist
    recv = torch.empty(sum(lay.recv_counts(g)), dtype=send.dtype, device=send.device)
    dist.all_to_all_single(recv, send, output_split_sizes=lay.recv_counts(g),
                           input_split_sizes=lay.send_counts(g), group=group)
    # span planes: all_gather wants equal sizes, shards may differ by one rank: pad the columns to the widest
    rows = lay.T * (lay.P + 1)
    rmax = max(r1 - r0 for r0, r1 in lay.ranks)
    rg = lay.ranks[g][1] - lay.ranks[g][0]
    mine = torch.zeros(rows, rmax, dtype=span_part.dtype, device=span_part.device)
    mine[:, :rg] = span_part.view(rows, rg)
    got = torch.empty(lay.G * rows * rmax, dtype=span_part.dtype, device=span_part.device)
    dist.all_gather_into_tensor(got, mine.view(-1), group=group)
    got = got.view(lay.G, rows, rmax)
    parts = [got[i, :, : r1 - r0].contiguous() for i, (r0, r1) in enumerate(lay.ranks)]
    return assemble_sig_plane(lay, g, recv), assemble_span_plane(lay, parts)


class PeerPlanes:
    """p2p exchange: every GPU's planes live in torch symmetric memory, so that a peer's pack kernel can
    store into them over NVLink.  Needs > 1 GPU with peer access: unmeasured on this pool's 1-GPU boxes
    (DESIGN.md §8); bench.py falls back to "a2a" when the rendezvous fails."""

    def __init__(self, lay: Layout, g: int, device: int, group_name: Optional[str] = None):
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm
        name = group_name or dist.group.WORLD.group_name
        smax = max(s1 - s0 for s0, s1 in lay.sigs)
        self.n_sig = lay.T * smax * lay.R
        self.n_span = lay.T * (lay.P + 1) * lay.R
        self.buf = symm.empty(self.n_sig + self.n_span, dtype=torch.int64, device=f"cuda:{device}")
        self.hdl = symm.rendezvous(self.buf, name)
        ptrs = list(self.hdl.buffer_ptrs)
        self.sig_ptrs = ptrs
        self.span_ptrs = [p + 8 * self.n_sig for p in ptrs]
        self.sig_plane = self.buf[: self.n_sig]
        self.span_plane = self.buf[self.n_sig:]

    def barrier(self):
        self.hdl.barrier()


# ---- bench.py --gpus N --scaling strong -------------------------------------------------------------------
def bench_strong(args, world, metric, measured_peak_gbs, ClockSampler, emit=True):
    """ONE job of the named workload over world.size GPUs: every GPU expands and aggregates its own ranks,
    one exchange, selection per sig slice.  Timed like the single-GPU step: CUDA events, max over ranks.
    emit=True: rank 0 prints the JSON line; emit=False: rank 0 returns it as a dict (the other ranks None), for
    bench.py's default N > 1 line, which carries the sharded job beside the weak-scaling headline."""
    import json
    import torch.distributed as dist
    from . import dist as D
    from .workload import build_workload
    G, g = world.size, world.rank
    dev = world.local_rank
    torch.cuda.set_device(dev)
    wl = build_workload(args.workload)
    s = wl.spec
    if s.shuffle:
        raise SystemExit("bench.py --scaling strong: the shuffled workload is not rank-partitioned")
    lay = Layout(G, s.n_ranks, s.n_steps, s.n_sigs, s.n_phases)
    sh = Shard(lay, g, s.step_base, device=dev)
    d_ev = wl.expand_device(sh.r0, sh.r1, device=f"cuda:{dev}")
    n = (sh.r1 - sh.r0) * s.n_steps * s.n_events
    # the shard's ctx addresses ranks relative to r0: rebase the rank field in place (input preparation)
    d_ev.view(torch.int32).view(-1, 8)[:, 0] -= sh.r0
    mode = args.exchange
    peer = None
    local = None
    if G == 1:
        # a world of one: the "exchange" is the pack kernel writing this GPU's own planes (the p2p path with
        # the local pointers) — runs the whole sharded step on a single-GPU box
        mode = "local"
        local = (torch.empty(lay.T * lay.S * lay.R, dtype=torch.int64, device=f"cuda:{dev}"),
                 torch.empty(lay.T * (lay.P + 1) * lay.R, dtype=torch.int64, device=f"cuda:{dev}"))
    elif mode == "p2p":
        try:
            peer = PeerPlanes(lay, g, dev)
        except Exception as e:                      # no peer access / symmetric memory on this box
            mode = "a2a"
            if g == 0:
                print(f"bench.py: p2p exchange unavailable ({repr(e)[:120]}); using all_to_all", flush=True)

    def step():
        sh.aggregate(d_ev, n)
        if local is not None:
            sh.pack_into_planes([local[0].data_ptr()], [local[1].data_ptr()])
            sh.diagnose(local[0], local[1])
            return
        if peer is not None:
            peer.barrier()                          # nobody still reads last step's planes
            sh.pack_into_planes(peer.sig_ptrs, peer.span_ptrs)
            peer.barrier()
            sig_plane, span_plane = peer.sig_plane, peer.span_plane
        else:
            sh.pack_for_all_to_all()
            sig_plane, span_plane = exchange_all_to_all(lay, g, sh.send, sh.span_part)
        sh.diagnose(sig_plane, span_plane)
        dist.all_reduce(sh.outs["rank_score"])       # partial HIGH counts -> straggler score of every rank

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    D.barrier(world)
    sampler = ClockSampler(dev).begin()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        step()
    b.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    D.barrier(world)
    ms_step = D.max_over_ranks(world, a.elapsed_time(b)) / args.steps
    nv, ni = sh.ctx.stats()
    total = D.sum_over_ranks(world, float(n))
    valid = D.sum_over_ranks(world, float(nv))
    sh.close()                                       # every rank releases its context, not only the one that prints
    if g != 0:
        return None
    peak, peak_src = measured_peak_gbs()
    table_bytes = s.n_ranks * s.n_steps * (64 + 32 * (s.n_phases + 1) + 160 * s.n_sigs)
    step_bytes = 32 * total + table_bytes
    line = {
        "metric": metric, "value": total / (ms_step * 1e-3), "unit": "events/s", "n_gpus": G,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": s.name, "n_ranks": s.n_ranks, "n_steps": s.n_steps,
                   "events_per_rank_step": s.n_events, "n_sigs": s.n_sigs, "n_phases": s.n_phases,
                   "events": int(total), "sharding": f"trace ranks over {G} GPUs, sig slices for the selection",
                   "exchange": mode, "exchange_bytes_total": 8 * s.n_ranks * s.n_steps * s.n_sigs,
                   "l2": "inputs (raw events) are larger than L2; no flush needed"},
        "raw_event_gbs": 32 * total / (ms_step * 1e-3) / 1e9,
        "hbm_frac_step_aggregate": step_bytes / (ms_step * 1e-3) / 1e9 / (peak * G),
        "roofline": None, "clocks": clocks, "e2e": None,
        "counters": {"n_valid": int(valid), "n_events": int(total)},
    }
    if emit:
        print(json.dumps(line))
    return line
