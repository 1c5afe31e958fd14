"""Seeded synthetic workloads shaped like the paper's kernel-event streams.

Input generator only — it serves both the CPU oracle tests and the CUDA path with the same event
bytes and holds none of the method's arithmetic.  All floating point happens HERE, once, when the
lookup tables are built; the expander that turns tables into 32-byte records is integer only and
exists as one source (expand_core.h) built for the host (gcc) and for the device (nvcc).

The five named workloads are BASELINE.json `configs[0..4]`; they stand in for the paper's
production traces, which are not public.
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import statistics
from typing import List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

EVENT_DTYPE = np.dtype(
    [("rank", "<u4"), ("step", "<u4"), ("sig", "<u4"), ("stream", "<u2"), ("phase", "<u2"),
     ("start_ns", "<i8"), ("end_ns", "<i8")])
assert EVENT_DTYPE.itemsize == 32

ANY = 0xFFFFFFFF
CLASS_COMM, CLASS_GEMM, CLASS_ATTN, CLASS_ELEM = 0, 1, 2, 3


def sig_class(sig: int) -> int:
    """Signature classes of the recipe: comm = sig < 32, else by sig mod 4."""
    if sig < 32:
        return CLASS_COMM
    m = sig & 3
    return CLASS_GEMM if m == 0 else (CLASS_ATTN if m == 1 else CLASS_ELEM)


@dataclasses.dataclass
class Fault:
    rank: int
    mult: float
    step: int = ANY        # relative step index
    sig: int = ANY
    sig_class: int = ANY
    phase: int = ANY

    def matches(self, t: int, sig: int, phase: int) -> bool:
        return ((self.step == ANY or self.step == t) and (self.sig == ANY or self.sig == sig)
                and (self.sig_class == ANY or self.sig_class == sig_class(sig))
                and (self.phase == ANY or self.phase == phase))


@dataclasses.dataclass
class Spec:
    name: str
    n_ranks: int
    n_steps: int
    n_events: int          # per rank-step
    n_sigs: int
    n_phases: int
    n_streams: int
    sig_dist: str          # "uniform" | "zipf"
    zipf_s: float
    mu_ns: float           # median base duration
    sigma: float           # log-normal sigma of per-sig base durations
    dur_mode: int = 0      # 0 lognormal base*jitter, 1 Pareto(1.5, xmin) per event
    shuffle: bool = False
    seed: int = 0
    step_base: int = 0
    fault_plan: str = ""   # which injected-fault recipe to use
    bimodal_frac: float = 0.0      # stress knob: this share of the sigs has a second duration mode ...
    bimodal_ratio: tuple = (8.0, 64.0)   # ... log-uniform in this range times the first, hit by half the events

    @property
    def total_events(self) -> int:
        return self.n_ranks * self.n_steps * self.n_events


_SEED0 = 260620374

CONFIGS = {
    # BASELINE.json configs[0]
    "tiny": Spec("tiny", 8, 4, 2000, 64, 4, 2, "uniform", 0.0, 20e3, 1.0, seed=_SEED0 + 0,
                 step_base=100, fault_plan="tiny"),
    # configs[1]
    "mid": Spec("mid", 256, 10, 20000, 512, 8, 4, "zipf", 1.1, 50e3, 1.2, seed=_SEED0 + 1,
                step_base=7, fault_plan="mid"),
    # configs[2] (P, streams not stated: as Mid)
    "scale": Spec("scale", 4096, 1, 80000, 1024, 8, 4, "zipf", 1.1, 50e3, 1.2, seed=_SEED0 + 2,
                  fault_plan="scale"),
    # configs[3] (P, streams not stated: as Mid)
    "unsorted": Spec("unsorted", 1024, 4, 50000, 2048, 8, 4, "uniform", 0.0, 5e3, 0.0, dur_mode=1,
                     shuffle=True, seed=_SEED0 + 3),
    # configs[4]
    "production": Spec("production", 4096, 1, 327680, 4096, 16, 8, "zipf", 1.05, 50e3, 1.2,
                       seed=_SEED0 + 4, fault_plan="production"),
}


def scaled(name: str, **kw) -> Spec:
    """A named config with some dimensions overridden (test-sized variants)."""
    s = dataclasses.replace(CONFIGS[name], **kw)
    s.name = name + "-scaled"
    return s


def _plan_faults(spec: Spec, rng: np.random.Generator) -> List[Fault]:
    R, S = spec.n_ranks, spec.n_sigs
    plan = spec.fault_plan
    if plan == "tiny":
        f = []
        if R > 5 and S > 17:
            f.append(Fault(rank=5, mult=1.5, sig=17))
        if R > 3 and spec.n_steps > 2 and spec.n_phases > 1:
            f.append(Fault(rank=3, mult=2.0, step=2, phase=1))
        return f
    if plan == "mid":
        k = min(3, R)
        ranks = rng.choice(R, size=k, replace=False)
        f = [Fault(rank=int(r), mult=1.3, sig_class=CLASS_GEMM) for r in ranks[:2]]
        if k > 2:
            f.append(Fault(rank=int(ranks[2]), mult=2.0, sig_class=CLASS_COMM))
        return f
    if plan == "scale":
        k = min(8, R)
        ranks = rng.choice(R, size=k, replace=False)
        return [Fault(rank=int(r), mult=1.2, sig_class=i % 4) for i, r in enumerate(ranks)]
    if plan == "production":
        k = min(16, R)
        ranks = rng.choice(R, size=min(R, k + 32), replace=False)
        f = [Fault(rank=int(r), mult=1.2, sig_class=i % 4) for i, r in enumerate(ranks[:k])]
        rest = ranks[k:]
        sigs = rng.choice(S, size=min(4, S), replace=False)
        for i, s in enumerate(sigs):
            for r in rest[8 * i: 8 * i + 8]:
                f.append(Fault(rank=int(r), mult=2.0, sig=int(s)))
        return f
    return []


class _FaultC(ctypes.Structure):
    _fields_ = [("rank", ctypes.c_uint32), ("step", ctypes.c_uint32), ("sig", ctypes.c_uint32),
                ("sig_class", ctypes.c_uint32), ("phase", ctypes.c_uint32),
                ("mult_q16", ctypes.c_uint32)]


FAULT_DTYPE = np.dtype([("rank", "<u4"), ("step", "<u4"), ("sig", "<u4"), ("sig_class", "<u4"),
                        ("phase", "<u4"), ("mult_q16", "<u4")])


class DescC(ctypes.Structure):
    """Mirror of wl_desc (expand_core.h)."""
    _fields_ = [("seed", ctypes.c_uint64),
                ("n_ranks", ctypes.c_uint32), ("n_steps", ctypes.c_uint32),
                ("n_events", ctypes.c_uint32), ("n_sigs", ctypes.c_uint32),
                ("n_phases", ctypes.c_uint32), ("n_streams", ctypes.c_uint32),
                ("step_base", ctypes.c_uint32), ("dur_mode", ctypes.c_uint32),
                ("shuffle", ctypes.c_uint32), ("n_faults", ctypes.c_uint32),
                ("xmin_ns", ctypes.c_uint64), ("step_gap_ns", ctypes.c_uint64),
                ("prog_sig", ctypes.c_void_p), ("prog_off", ctypes.c_void_p),
                ("stream_id", ctypes.c_void_p), ("base_ns", ctypes.c_void_p),
                ("jit_q16", ctypes.c_void_p), ("gap_ns", ctypes.c_void_p),
                ("pareto_q16", ctypes.c_void_p), ("faults", ctypes.c_void_p),
                ("fault_off", ctypes.c_void_p), ("mode2_q16", ctypes.c_void_p)]


_TABLE_NAMES = ["prog_sig", "prog_off", "stream_id", "base_ns", "jit_q16", "gap_ns", "pareto_q16",
                "faults", "fault_off", "mode2_q16"]


class Workload:
    """Tables of one seeded workload + the two expanders (host C, device CUDA)."""

    def __init__(self, spec: Spec):
        if not (1 <= spec.n_streams <= 16):
            raise ValueError("n_streams must be 1..16")
        self.spec = spec
        rng = np.random.Generator(np.random.PCG64(spec.seed))
        S, N, T, J = spec.n_sigs, spec.n_events, spec.n_steps, spec.n_streams
        nd = statistics.NormalDist()

        # per-sig base duration: lognormal(ln mu, sigma) (BASELINE.json configs)
        z = rng.standard_normal(S)
        base = np.maximum(1, np.rint(spec.mu_ns * np.exp(spec.sigma * z))).astype(np.uint64)
        # per-event jitter lognormal(0, 0.1) and exponential gaps (mean 2 us) as quantile tables
        q = (np.arange(4096) + 0.5) / 4096.0
        jit = np.array([round(65536.0 * math.exp(0.1 * nd.inv_cdf(float(u)))) for u in q],
                       dtype=np.uint32)
        gap = np.array([round(-2000.0 * math.log(1.0 - float(u))) for u in q], dtype=np.uint32)
        # Pareto(alpha=1.5) ratio quantiles; the top cell chains a second draw (self-similar tail)
        q16 = (np.arange(65536) + 0.5) / 65536.0
        par = np.rint(65536.0 * (1.0 - q16) ** (-1.0 / 1.5)).astype(np.uint32)

        # step program shared by all ranks: sigs per step, grouped by stream
        if spec.sig_dist == "zipf":
            w = 1.0 / np.arange(1, S + 1, dtype=np.float64) ** spec.zipf_s
            p = w / w.sum()
            perm = rng.permutation(S)          # popularity rank -> sig id ("hot" ids unpredictable)
        else:
            p = np.full(S, 1.0 / S)
            perm = np.arange(S)
        self.sig_popularity_perm = perm
        prog = np.empty((T, N), dtype=np.uint32)
        off = np.zeros((T, J + 1), dtype=np.uint32)
        for t in range(T):
            sigs = perm[rng.choice(S, size=N, p=p)].astype(np.uint32)
            if J == 1:
                strm = np.zeros(N, dtype=np.int64)
            else:
                strm = np.where(sigs < 32, J - 1, sigs % (J - 1)).astype(np.int64)
            order = np.argsort(strm, kind="stable")
            prog[t] = sigs[order]
            off[t, 1:] = np.cumsum(np.bincount(strm, minlength=J))
        stream_id = np.array([7 + j for j in range(J)], dtype=np.uint16)
        if J > 1:
            stream_id[J - 1] = 31               # the comm stream (e.g. 7 and 31)

        self.faults: List[Fault] = sorted(_plan_faults(spec, rng), key=lambda f: f.rank)
        fa = np.zeros(max(1, len(self.faults)), dtype=FAULT_DTYPE)
        foff = np.zeros(spec.n_ranks + 1, dtype=np.uint32)
        for i, f in enumerate(self.faults):
            fa[i] = (f.rank, f.step, f.sig, f.sig_class, f.phase, round(f.mult * 65536))
            foff[f.rank + 1:] += 1

        # stress knob (bench.py --bimodal): a second duration mode for a share of the sigs, drawn from
        # its own generator so that the named workloads keep their bytes
        mode2 = np.zeros(S, dtype=np.uint32)
        if spec.bimodal_frac > 0.0:
            rng2 = np.random.Generator(np.random.PCG64(spec.seed ^ 0x5EED))
            pick = rng2.random(S) < spec.bimodal_frac
            lo, hi = spec.bimodal_ratio
            ratio = np.exp(rng2.uniform(math.log(lo), math.log(hi), size=S))
            mode2[pick] = np.rint(65536.0 * ratio[pick]).astype(np.uint32)
        self.n_bimodal = int((mode2 != 0).sum())

        self.tables = dict(prog_sig=prog.reshape(-1), prog_off=off.reshape(-1), stream_id=stream_id,
                           base_ns=base, jit_q16=jit, gap_ns=gap, pareto_q16=par, faults=fa,
                           fault_off=foff, mode2_q16=mode2)
        self._dev_tables = None
        self._host_lib = None
        self._dev_lib = None

    # ---- descriptors ----------------------------------------------------------------------
    def _desc(self, ptrs) -> DescC:
        s = self.spec
        d = DescC()
        d.seed = s.seed
        d.n_ranks, d.n_steps, d.n_events = s.n_ranks, s.n_steps, s.n_events
        d.n_sigs, d.n_phases, d.n_streams = s.n_sigs, s.n_phases, s.n_streams
        d.step_base, d.dur_mode, d.shuffle = s.step_base, s.dur_mode, int(s.shuffle)
        d.n_faults = len(self.faults)
        d.xmin_ns = int(s.mu_ns)
        d.step_gap_ns = 50_000
        for k in _TABLE_NAMES:
            setattr(d, k, ptrs[k])
        return d

    def manifest(self) -> dict:
        s = self.spec
        return dict(name=s.name, seed=s.seed, n_ranks=s.n_ranks, n_steps=s.n_steps,
                    n_events=s.n_events, n_sigs=s.n_sigs, n_phases=s.n_phases,
                    n_streams=s.n_streams, step_base=s.step_base, shuffle=s.shuffle,
                    dur_mode=s.dur_mode, faults=[dataclasses.asdict(f) for f in self.faults])

    # ---- host expander ---------------------------------------------------------------------
    def expand_host(self, rank_lo: int = 0, rank_hi: Optional[int] = None,
                    threads: Optional[int] = None, out: Optional[np.ndarray] = None) -> np.ndarray:
        """Events of ranks [rank_lo, rank_hi) as an EVENT_DTYPE array.  With shuffle the result is
        the FULL buffer (all ranks must be expanded for it to be complete)."""
        from .build import load_host_lib
        s = self.spec
        rank_hi = s.n_ranks if rank_hi is None else rank_hi
        if self._host_lib is None:
            self._host_lib = load_host_lib()
        n = s.total_events if s.shuffle else (rank_hi - rank_lo) * s.n_steps * s.n_events
        if out is None:
            out = np.zeros(n, dtype=EVENT_DTYPE)
        assert out.dtype == EVENT_DTYPE and out.size == n and out.flags.c_contiguous
        d = self._desc({k: v.ctypes.data for k, v in self.tables.items()})
        threads = threads or min(32, os.cpu_count() or 1)
        rc = self._host_lib.wl_expand_host(ctypes.byref(d), rank_lo, rank_hi,
                                           ctypes.c_void_p(out.ctypes.data), threads)
        if rc != 0:
            raise RuntimeError(f"wl_expand_host failed: {rc}")
        return out

    # ---- device expander -------------------------------------------------------------------
    def expand_device(self, rank_lo: int = 0, rank_hi: Optional[int] = None, out=None,
                      device: str = "cuda:0"):
        """Same bytes as expand_host, written straight into HBM (torch uint8 tensor)."""
        import torch
        from .build import load_device_lib
        s = self.spec
        rank_hi = s.n_ranks if rank_hi is None else rank_hi
        if self._dev_lib is None:
            self._dev_lib = load_device_lib()
        if self._dev_tables is None:
            self._dev_tables = {
                k: torch.from_numpy(v.view(np.uint8).reshape(-1).copy()).to(device)
                for k, v in self.tables.items()}
        n = s.total_events if s.shuffle else (rank_hi - rank_lo) * s.n_steps * s.n_events
        if out is None:
            out = torch.empty(n * 32, dtype=torch.uint8, device=device)
        assert out.numel() == n * 32 and out.is_cuda and out.is_contiguous()
        d = self._desc({k: v.data_ptr() for k, v in self._dev_tables.items()})
        stream = torch.cuda.current_stream(out.device).cuda_stream
        with torch.cuda.device(out.device):
            rc = self._dev_lib.wl_expand_device(ctypes.byref(d), rank_lo, rank_hi,
                                                ctypes.c_void_p(out.data_ptr()),
                                                ctypes.c_void_p(stream))
        if rc != 0:
            raise RuntimeError(f"wl_expand_device failed: {rc}")
        return out


def build_workload(name_or_spec) -> Workload:
    spec = CONFIGS[name_or_spec] if isinstance(name_or_spec, str) else name_or_spec
    return Workload(spec)
