"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default
kernel geometry, one argus_aggregate over the whole resident buffer): every byte of the record
table and of the diagnosis is compared with the CPU oracle, which consumes the same seeded events
expanded on the host chunk by chunk (the device buffer is written by the device build of the same
integer expander; test_device_expander_matches_host pins the two builds to each other, and the
n_valid / n_invalid counters and every record byte pin them again here)."""
import time

import numpy as np
import pytest

from gpu_util import first_diff
from oracle import Oracle
from paper_2606_20374_b200.workload import build_workload

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def _full_parity(name, chunk_ranks):
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(name)
    s = wl.spec
    free, _ = torch.cuda.mem_get_info()
    need = s.total_events * 32 * (2 if s.shuffle else 1) + \
        s.n_ranks * s.n_steps * (64 + 32 * (s.n_phases + 1) + 168 * s.n_sigs)
    if free < need * 1.05:
        pytest.skip(f"{name}: needs {need / 1e9:.1f} GB of HBM, {free / 1e9:.1f} GB free")
    # ---- CUDA path, as bench.py runs it ----------------------------------------------------------
    d_ev = wl.expand_device()
    ctx = A.Argus(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base, sorted_hint=not s.shuffle,
                  max_ungrouped_events=s.total_events if s.shuffle else 0)
    rec = ctx.alloc_records()
    outs = ctx.alloc_diag()
    ctx.reset(rec)
    ctx.aggregate(d_ev, s.total_events, rec)
    ctx.phase_times(rec)
    ctx.diagnose(rec, outs)
    stats = ctx.stats()
    del d_ev
    got_rec = ctx.records_to_host(rec)
    got = ctx.diag_to_host(outs)
    ctx.close()
    del rec, outs
    torch.cuda.empty_cache()
    # ---- oracle on the host expansion of the same workload -------------------------------------------
    t0 = time.time()
    o = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    if s.shuffle:
        o.aggregate(wl.expand_host())
    else:
        for lo in range(0, s.n_ranks, chunk_ranks):
            o.aggregate(wl.expand_host(lo, min(s.n_ranks, lo + chunk_ranks)))
    assert stats == (o.n_valid, o.n_invalid) == (s.total_events, 0)
    want_rec = o.records()
    if not np.array_equal(got_rec, want_rec):
        i = first_diff(got_rec, want_rec)
        rb = got_rec.shape[1]
        raise AssertionError(f"{name}: records differ at record {i // rb} offset {i % rb}")
    del want_rec, got_rec
    want = o.diagnose()
    for k in ("sig_stats", "sig_flags", "span_stats", "span_flags", "rank_score", "step_anomalous"):
        assert np.array_equal(got[k], want[k]), (name, k)
    # injected stragglers stand out: class-wide fault ranks top the HIGH counts of their class
    # (comm-class faults touch only sigs < 32, so they are ranked on those sigs alone)
    wide = [f for f in wl.faults if f.sig == 0xFFFFFFFF and f.phase == 0xFFFFFFFF]
    for comm in (False, True):
        ranks = sorted({f.rank for f in wide if (f.sig_class == 0) == comm})
        if ranks:
            fl = want["sig_flags"][:, :32] if comm else want["sig_flags"][:, 32:]
            score = (fl == 1).sum(axis=(0, 1)).astype(np.int64)
            top = set(np.argsort(-score, kind="stable")[: len(ranks)].tolist())
            assert top == set(ranks), (name, comm, ranks, sorted(top))
    print(f"{name}: {s.total_events} events bit-exact, oracle side {time.time() - t0:.0f} s")


def test_mid_full_size():
    _full_parity("mid", 64)


def test_scale_full_size():
    _full_parity("scale", 512)


def test_unsorted_full_size():
    _full_parity("unsorted", 0)


def test_production_full_size():
    _full_parity("production", 128)
