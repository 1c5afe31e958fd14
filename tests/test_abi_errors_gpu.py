"""-m gpu tests of the boundary's error behaviour and call-order rules (SURVEY §8(b) "Errors";
include/argus.h): negative codes, never exceptions or faults; no allocation after argus_create."""
import ctypes

import numpy as np
import pytest

from gpu_util import compare_with_oracle
from helpers import make_events
from paper_2606_20374_b200.workload import build_workload, scaled

pytestmark = pytest.mark.gpu


def _dims(spec):
    return spec.n_ranks, spec.n_steps, spec.n_sigs, spec.n_phases, spec.step_base


def _dev(ev):
    import torch
    raw = np.ascontiguousarray(ev).view(np.uint8).reshape(-1)
    return torch.from_numpy(raw.copy()).cuda()


def _code(fn, *a, **k):
    from paper_2606_20374_b200 import argus as A
    try:
        fn(*a, **k)
    except A.ArgusError as e:
        return e.code
    return A.OK


def test_call_order_and_argument_errors():
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("tiny", n_ranks=3, n_steps=2, n_events=700))
    ev = wl.expand_host()
    d_ev = _dev(ev)
    ctx = A.Argus(*_dims(wl.spec))
    rec, other = ctx.alloc_records(), ctx.alloc_records()
    outs = ctx.alloc_diag()
    # nothing was reset yet: every table is foreign
    assert _code(ctx.aggregate, d_ev, ev.size, rec) == A.ESTATE
    assert _code(ctx.phase_times, rec) == A.ESTATE
    ctx.reset(rec)
    assert _code(ctx.aggregate, d_ev, ev.size, other) == A.ESTATE       # not the table given to reset
    assert _code(ctx.aggregate_host, None, 0, 1, None, 0, other) == A.ESTATE
    assert _code(ctx.phase_times, other) == A.ESTATE
    assert _code(ctx.diagnose, rec, outs) == A.ESTATE                   # own table, not finalised
    # argument errors
    assert _code(ctx.aggregate, d_ev.data_ptr() + 8, 10, rec) == A.EINVAL      # misaligned events
    assert _code(ctx.aggregate, None, 10, rec) == A.EINVAL
    assert _code(ctx.aggregate, d_ev, 1 << 32, rec) == A.ESIZE
    assert _code(ctx.reset, rec.data_ptr() + 4) == A.EINVAL
    assert _code(ctx.reset, None) == A.EINVAL
    assert _code(ctx.phase_times, rec, rec.data_ptr() + 8) == A.EINVAL         # misaligned spans_out
    assert _code(ctx.diagnose, rec.data_ptr() + 8, outs) == A.EINVAL
    bad = dict(outs)
    bad["sig_stats"] = outs["sig_stats"].data_ptr() + 8
    assert _code(ctx.diagnose, other, bad) == A.EINVAL
    bad = dict(outs)
    bad["rank_score"] = outs["rank_score"].data_ptr() + 2
    assert _code(ctx.diagnose, other, bad) == A.EINVAL
    assert _code(ctx.tune, 99, 0) == A.EINVAL and _code(ctx.tune, A.TUNE_GRID_CTAS, 1025) == A.EINVAL
    assert _code(ctx.tune, A.TUNE_FORCE_PATH, 4) == A.EINVAL
    lib = ctx.lib
    assert lib.argus_stats(None, None, None) == A.EINVAL
    assert lib.argus_stats(ctx._h, None, None) == A.OK                  # NULL outputs are allowed
    # the failed calls left the ctx usable: the plain sequence still matches the oracle
    ctx.reset(rec)
    ctx.aggregate(d_ev, ev.size, rec)
    ctx.aggregate(None, 0, rec)                                          # n = 0 needs no pointer
    assert _code(ctx.diagnose, rec, outs) == A.ESTATE
    ctx.phase_times(rec)
    ctx.diagnose(rec, outs)
    compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), ctx.stats(), None, ev, *_dims(wl.spec))
    ctx.close()


def test_workspace_ownership_and_no_allocation_after_create():
    """the caller owns every large buffer.  Between argus_create and argus_destroy the
    library allocates nothing on the device and never synchronises it: cudaMemGetInfo is unchanged
    across reset / aggregate (grouped, ungrouped, host-streamed) / phase_times / diagnose."""
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("unsorted", n_ranks=16, n_events=5000))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    n = ev.size
    d_ev = _dev(ev)
    h = torch.empty(n * 32, dtype=torch.uint8, pin_memory=True)
    h.copy_(d_ev)
    ring = torch.empty(2 * 50_000 * 32, dtype=torch.uint8, device="cuda")
    for ws in ("torch", None):
        ctx = A.Argus(*dims[:4], dims[4], sorted_hint=False, max_ungrouped_events=n, workspace=ws)
        assert ctx.workspace_bytes >= 8 * dims[0] * dims[1] * dims[2] + 32 * n     # sum plane + grouping area
        if ws == "torch":
            assert ctx.workspace.numel() == ctx.workspace_bytes
        rec = ctx.alloc_records()
        outs = ctx.alloc_diag()
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for path in (0, A.PATH_SEGMENTED, A.PATH_GLOBAL):
            ctx.tune(A.TUNE_FORCE_PATH, path)
            ctx.reset(rec)
            ctx.aggregate(d_ev, n // 2, rec)
            ctx.aggregate_host(h.data_ptr() + (n // 2) * 32, n - n // 2, 50_000, ring, 2, rec)
            ctx.phase_times(rec)
            ctx.diagnose(rec, outs)
            assert torch.cuda.mem_get_info()[0] == free0
            compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), ctx.stats(), None, ev, *dims)
        # a call larger than the grouping area takes the global-table kernel (no allocation either)
        small = A.Argus(*dims[:4], dims[4], sorted_hint=False, max_ungrouped_events=1000, workspace=ws)
        small.reset(rec)
        small.aggregate(d_ev, n, rec)
        small.phase_times(rec)
        small.diagnose(rec, outs)
        compare_with_oracle(small.records_to_host(rec), small.diag_to_host(outs), small.stats(), None, ev, *dims)
        small.close()
        ctx.close()
    # a workspace that is too small, or misaligned, is refused
    cfg = A.ArgusConfig(*dims[:4], dims[4], 0, 0, n)
    lib = A.load()
    need = lib.argus_workspace_bytes(ctypes.byref(cfg))
    buf = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    hnd = ctypes.c_void_p()
    assert lib.argus_create(ctypes.byref(cfg), buf.data_ptr(), need - 1, ctypes.byref(hnd)) == A.EINVAL
    assert lib.argus_create(ctypes.byref(cfg), buf.data_ptr() + 16, need, ctypes.byref(hnd)) == A.EINVAL
    assert lib.argus_create(ctypes.byref(cfg), buf.data_ptr(), need, ctypes.byref(hnd)) == A.OK
    assert lib.argus_destroy(hnd) == A.OK


def test_advertised_sequence_aggregate_finalise_twice():
    """argus.h: argus_phase_times is idempotent and "may be followed by more argus_aggregate calls and
    another argus_phase_times".  aggregate -> phase_times -> aggregate -> phase_times -> diagnose equals
    the oracle over all events; the intermediate table equals the oracle over the first part."""
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("mid", n_ranks=10, n_steps=2, n_events=6000))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    d_ev = _dev(ev)
    cut = 47_001                                     # inside a rank-step; ranks 8, 9 untouched so far
    ctx = A.Argus(*dims)
    rec = ctx.alloc_records()
    rec.fill_(0xAB)
    outs = ctx.alloc_diag()
    ctx.reset(rec)
    ctx.aggregate(d_ev, cut, rec)
    ctx.phase_times(rec)
    ctx.phase_times(rec)                             # idempotent
    ctx.diagnose(rec, outs)
    compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), ctx.stats(), None, ev[:cut], *dims)
    ctx.aggregate(d_ev.data_ptr() + cut * 32, ev.size - cut, rec)
    assert _code(ctx.diagnose, rec, outs) == A.ESTATE       # stale span_ns / headers are never diagnosed
    ctx.phase_times(rec)
    ctx.diagnose(rec, outs)
    compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), ctx.stats(), None, ev, *dims)
    ctx.close()


def test_null_outputs_are_skipped():
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("tiny", n_ranks=5, n_steps=2, n_events=900))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    d_ev = _dev(ev)
    ctx = A.Argus(*dims)
    rec = ctx.alloc_records()
    ctx.reset(rec)
    ctx.aggregate(d_ev, ev.size, rec)
    ctx.phase_times(rec)
    full = ctx.alloc_diag()
    ctx.diagnose(rec, full)
    want = ctx.diag_to_host(full)
    names = list(full)
    for keep in (["sig_flags"], ["rank_score"], ["span_stats", "step_anomalous"], ["sig_stats", "span_flags"], []):
        outs = ctx.alloc_diag()
        for v in outs.values():
            v.fill_(0x5A if v.dtype == torch.uint8 else 0x5A5A5A5A)
        ctx.diagnose(rec, {k: outs[k] for k in keep})
        got = ctx.diag_to_host(outs)
        for k in names:
            if k in keep:
                assert (got[k] == want[k]).all(), (keep, k)
            else:                                   # untouched: still the fill pattern
                assert (got[k].view(np.uint8) == 0x5A).all(), (keep, k)
    ctx.close()


def test_step_base_at_the_top_of_u32():
    """step numbers do not wrap.  step_base + T == 2^32 is the last legal window; events of
    steps 0, 1 (which would alias t = 4, 5 mod 2^32 in a wider window) are invalid, as in the oracle."""
    base = 2**32 - 4
    rows = []
    for r in range(3):
        for t in range(4):
            for i in range(40):
                rows.append((r, base + t, i % 5, 0, i % 2, 1000 * i, 1000 * i + 100 + r + t))
        rows += [(r, 0, 1, 0, 0, 5, 50), (r, 1, 2, 0, 1, 5, 60), (r, base - 1, 0, 0, 0, 5, 70)]
    ev = make_events(rows)
    import torch
    from paper_2606_20374_b200 import argus as A
    for hint, path in ((True, 1), (True, 2), (False, 0)):
        ctx = A.Argus(3, 4, 5, 2, base, sorted_hint=hint, max_ungrouped_events=ev.size)
        ctx.tune(A.TUNE_FORCE_PATH, path)
        rec = ctx.alloc_records()
        outs = ctx.alloc_diag()
        ctx.reset(rec)
        ctx.aggregate(_dev(ev), ev.size, rec)
        ctx.phase_times(rec)
        ctx.diagnose(rec, outs)
        stats = ctx.stats()
        assert stats == (480, 9)
        compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), stats, None, ev, 3, 4, 5, 2, base)
        ctx.close()
    with pytest.raises(A.ArgusError) as e:
        A.Argus(3, 5, 5, 2, base)
    assert e.value.code == A.ESIZE


def test_launch_count_is_counted_not_assumed():
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("tiny", n_ranks=2, n_steps=1, n_events=300))
    ev = wl.expand_host()
    ctx = A.Argus(*_dims(wl.spec))
    rec = ctx.alloc_records()
    outs = ctx.alloc_diag()
    assert ctx.launch_count() == (0, 0)
    ctx.reset(rec)
    assert ctx.launch_count() == (0, 1)
    ctx.aggregate(_dev(ev), ev.size, rec)
    k1 = ctx.launch_count()[0]
    assert k1 >= 1
    ctx.phase_times(rec)
    ctx.diagnose(rec, outs)
    k2, m2 = ctx.launch_count()
    assert k2 > k1 + 1 and m2 == 2                   # finalize + selection kernels; rank_score clear
    ctx.close()


def test_refused_count_diagnostic():
    """Events the compact shared-memory cell cannot hold are re-queued through the spill area (range wider
    than four buckets) or take the overflow list (>= 2^32 ns; everything when there is no spill area); both
    are counted, and the results are exact either way (compare_with_oracle)."""
    from paper_2606_20374_b200 import argus as A
    n = 20000
    # sig 0: one mode (no refusals); sig 1: two modes 2^10 and 2^20 (one of them is refused);
    # sig 2: durations >= 2^32 ns (no 32-bit cell can hold them)
    rows = []
    for i in range(n):
        rows.append((0, 0, 0, 0, 0, i, i + 1000 + i % 50))
        rows.append((0, 0, 1, 0, 0, i, i + ((1 << 10) + i % 7 if i % 2 else (1 << 20) + i % 5)))
        if i % 10 == 0:
            rows.append((0, 0, 2, 0, 0, i, i + (1 << 33) + i))
    ev = make_events(rows)
    for spill in (0, ev.size, 3000):
        ctx = A.Argus(1, 1, 3, 1, max_spill_events=spill)
        rec = ctx.alloc_records()
        outs = ctx.alloc_diag()
        ctx.reset(rec)
        ctx.aggregate(_dev(ev), ev.size, rec)
        ctx.phase_times(rec)
        ctx.diagnose(rec, outs)
        requeued, overflow = ctx.refused_count()
        if spill == 0:
            assert requeued == 0 and 0.45 * n + n // 10 <= overflow <= n + n // 10, (requeued, overflow)   # every CTA refuses one of the modes
        elif spill == ev.size:
            assert 0.45 * n <= requeued <= n and overflow == n // 10, (requeued, overflow)   # one mode of sig 1; all of sig 2
        else:
            assert 0 < requeued <= 3000 and overflow >= 0.45 * n + n // 10 - requeued, (requeued, overflow)   # the area ran out
        compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), ctx.stats(), None, ev, 1, 1, 3, 1, 0)
        ctx.reset(rec)
        ctx.aggregate(_dev(ev[ev["sig"] == 0]), n, rec)
        assert ctx.refused_count() == (0, 0)
        ctx.close()
