"""-m gpu parity tests of row a1 (NS (2): "an ingest path from pinned host chunks via cudaMemcpyAsync on
a side stream, overlapped with compute"; BASELINE.json configs[4]: "streamed from pinned host memory in
256 MB chunks overlapped with aggregation"; the paper's fixed buffer pool):
argus_aggregate_host and argus_ingest + argus_aggregate, every record byte and every diagnosis output
against the CPU oracle on the same seeded bytes."""
import numpy as np
import pytest

from gpu_util import compare_with_oracle
from paper_2606_20374_b200.workload import EVENT_DTYPE, build_workload, scaled

pytestmark = pytest.mark.gpu

PATH_SEG, PATH_GLOBAL, PATH_GROUPED = 1, 2, 3


def _dims(spec):
    return spec.n_ranks, spec.n_steps, spec.n_sigs, spec.n_phases, spec.step_base


def _pinned(ev):
    import torch
    raw = np.ascontiguousarray(ev).view(np.uint8).reshape(-1)
    h = torch.empty(max(raw.size, 32), dtype=torch.uint8, pin_memory=True)
    h[: raw.size].copy_(torch.from_numpy(raw.copy()))
    return h


def _finish(ctx, rec, ev, dims):
    """phase_times + diagnose, read back, compare everything with the oracle."""
    import torch
    from paper_2606_20374_b200 import argus as A
    R, T, S, P, base = dims
    spans_out = torch.empty(R * T * (P + 1) * 32, dtype=torch.uint8, device="cuda")
    ctx.phase_times(rec, spans_out)
    outs = ctx.alloc_diag()
    for v in outs.values():
        v.fill_(0x5A if v.dtype == torch.uint8 else 0x5A5A5A5A)
    ctx.diagnose(rec, outs)
    stats = ctx.stats()
    compare_with_oracle(ctx.records_to_host(rec), ctx.diag_to_host(outs), stats,
                        spans_out.cpu().numpy().view(A.SPAN_DTYPE).reshape(R, T, P + 1), ev, *dims)


def _run_host(ev, dims, chunk, slots, sorted_hint=True, path=None, repeat=1):
    import torch
    from paper_2606_20374_b200 import argus as A
    n = ev.size
    ctx = A.Argus(*dims[:4], dims[4], sorted_hint=sorted_hint,
                  max_ungrouped_events=0 if (sorted_hint and path != PATH_GROUPED) else chunk)
    if path is not None:
        ctx.tune(A.TUNE_FORCE_PATH, path)
    h = _pinned(ev)
    ring = torch.empty(slots * chunk * 32, dtype=torch.uint8, device="cuda")
    rec = ctx.alloc_records()
    for _ in range(repeat):           # a second pass re-uses the ring right behind the first one's tail
        ring.fill_(0xCD)              # garbage: a chunk aggregated before its copy landed would show
        rec.fill_(0xAB)
        ctx.reset(rec)
        ctx.aggregate_host(h, n, chunk, ring, slots, rec)
    _finish(ctx, rec, ev, dims)
    ctx.close()


@pytest.mark.parametrize("slots", [1, 2, 3])
def test_aggregate_host_ring_reuse(slots):
    # 64,000 events in chunks of 9,001 (not a multiple of 4: the ragged tail of the TMA tensor in every
    # chunk): 8 chunks > ring slots (slot reuse), a short last chunk (993), every chunk cuts a rank-step
    wl = build_workload("tiny")
    ev = wl.expand_host()
    _run_host(ev, _dims(wl.spec), 9001, slots, repeat=2)


@pytest.mark.parametrize("path", [PATH_GLOBAL, PATH_GROUPED])
def test_aggregate_host_other_paths(path):
    wl = build_workload("tiny")
    ev = wl.expand_host()
    _run_host(ev, _dims(wl.spec), 9001, 2, path=path)


def test_aggregate_host_ungrouped_input():
    # shuffled input without the SORTED hint through the host path: every chunk is grouped on its own
    wl = build_workload(scaled("unsorted", n_ranks=32, n_events=6000))
    ev = wl.expand_host()
    _run_host(ev, _dims(wl.spec), 100_003, 3, sorted_hint=False)


def test_aggregate_host_mid_scaled_chunks_cut_rank_steps():
    # mid-shaped (S = 512: three CTAs per SM), 12 ranks x 2 steps x 20,000 events in 11 chunks of 45,678
    wl = build_workload(scaled("mid", n_ranks=12, n_steps=2))
    ev = wl.expand_host()
    assert ev.size // 45_678 + 1 == 11
    _run_host(ev, _dims(wl.spec), 45_678, 3)


def test_aggregate_host_production_scaled():
    # S = 4,096 (one CTA per SM), chunk = 1 MiB of events, 2-slot ring
    wl = build_workload(scaled("production", n_ranks=6, n_events=50_001))
    ev = wl.expand_host()
    _run_host(ev, _dims(wl.spec), 32_768, 2)


def test_aggregate_host_empty_and_single_chunk():
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("tiny", n_ranks=2, n_steps=1, n_events=500))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    ctx = A.Argus(*dims[:4], dims[4])
    rec = ctx.alloc_records()
    rec.fill_(0xAB)
    ring = torch.empty(4096 * 32, dtype=torch.uint8, device="cuda")
    ctx.reset(rec)
    ctx.aggregate_host(None, 0, 4096, None, 0, rec)         # n = 0: nothing to do, nothing checked
    _finish(ctx, rec, ev[:0], dims)
    ctx.reset(rec)
    ctx.aggregate_host(_pinned(ev), ev.size, 4096, ring, 1, rec)   # one chunk shorter than a slot
    _finish(ctx, rec, ev, dims)
    # bad arguments
    h = _pinned(ev)
    for args in ((h, ev.size, 0, ring, 1), (h, ev.size, 4096, ring, 0), (h, ev.size, 4096, ring, 65),
                 (h, ev.size, 4096, None, 1), (None, ev.size, 4096, ring, 1)):
        with pytest.raises(A.ArgusError) as e:
            ctx.aggregate_host(*args, rec)
        assert e.value.code == A.EINVAL
    with pytest.raises(A.ArgusError) as e:
        ctx.aggregate_host(h, ev.size, 1 << 32, ring, 1, rec)
    assert e.value.code == A.ESIZE
    ctx.close()


@pytest.mark.parametrize("chunk", [7_777, 20_000])
def test_ingest_double_buffered(chunk):
    """argus_ingest on the caller's copy stream + argus_aggregate on a compute stream, two device
    buffers: the internal event must order every copy before the kernel that reads it (the buffers are
    filled with garbage first), and the caller's own event orders buffer re-use."""
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("mid", n_ranks=6, n_steps=2, n_events=10_000))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    n = ev.size
    h = _pinned(ev)
    ctx = A.Argus(*dims[:4], dims[4])
    rec = ctx.alloc_records()
    rec.fill_(0xAB)
    bufs = [torch.full((chunk * 32,), 0xCD, dtype=torch.uint8, device="cuda") for _ in range(2)]
    copy_s, comp_s = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    done = [None, None]                       # compute-stream event after the last kernel that read buf i
    ctx.reset(rec, stream=comp_s)
    for c, a in enumerate(range(0, n, chunk)):
        cnt = min(chunk, n - a)
        b = c % 2
        if done[b] is not None:
            copy_s.wait_event(done[b])        # buffer re-use is the caller's business (argus.h)
        ctx.ingest(h.data_ptr() + a * 32, cnt, bufs[b], copy_s)
        ctx.aggregate(bufs[b], cnt, rec, stream=comp_s)
        done[b] = torch.cuda.Event()
        done[b].record(comp_s)
    with torch.cuda.stream(comp_s):
        _finish(ctx, rec, ev, dims)
    ctx.close()


def test_ingest_then_aggregate_host_keeps_the_dependency():
    """an argus_ingest queued before argus_aggregate_host must stay ordered before the next
    kernel that reads its destination (the host path used to overwrite the pending event)."""
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("tiny", n_ranks=4, n_steps=2, n_events=4000))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    half = ev.size // 2
    h = _pinned(ev)
    ctx = A.Argus(*dims[:4], dims[4])
    rec = ctx.alloc_records()
    d_first = torch.full((half * 32,), 0xCD, dtype=torch.uint8, device="cuda")
    ring = torch.empty(2 * 3000 * 32, dtype=torch.uint8, device="cuda")
    copy_s = torch.cuda.Stream()
    torch.cuda.synchronize()
    ctx.reset(rec)
    ctx.ingest(h, half, d_first, copy_s)                                   # first half: caller's copy
    ctx.aggregate_host(h.data_ptr() + half * 32, ev.size - half, 3000, ring, 2, rec)   # second half: streamed
    ctx.aggregate(d_first, half, rec)                                      # must see the ingested bytes
    _finish(ctx, rec, ev, dims)
    ctx.close()


def test_host_to_host_events_in_summary_stream_out():
    """The whole e2e shape bench.py times (NS (2)-(5); the reducer's upload of its summaries):
    pinned host events -> argus_aggregate_host -> phase_times -> diagnose -> argus_sparse_encode -> the stream and
    its offsets copied to pinned HOST memory.  The host-side bytes, decoded by the independent reader of
    tests/helpers.py, must rebuild the oracle's table byte for byte."""
    import torch
    from gpu_util import run_oracle
    from helpers import sparse_to_dense
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("mid", n_ranks=12, n_steps=3, n_events=5000, n_sigs=300))
    ev = wl.expand_host()
    dims = _dims(wl.spec)
    R, T, S, P, base = dims
    chunk = 7777                                         # ragged: cuts rank-steps anywhere
    ctx = A.Argus(R, T, S, P, base)
    h = _pinned(ev)
    ring = torch.empty(2 * chunk * 32, dtype=torch.uint8, device="cuda")
    rec = ctx.alloc_records()
    rec.fill_(0xAB)
    ctx.reset(rec)
    ctx.aggregate_host(h, ev.size, chunk, ring, 2, rec)
    ctx.phase_times(rec)
    outs = ctx.alloc_diag()
    ctx.diagnose(rec, outs)
    d_out = torch.empty(ctx.sparse_bound(), dtype=torch.uint8, device="cuda")
    d_off = torch.zeros(R * T + 1, dtype=torch.int64, device="cuda")
    ctx.sparse_encode(rec, d_out, d_off)
    h_off = torch.empty(R * T + 1, dtype=torch.int64, pin_memory=True)
    h_off.copy_(d_off, non_blocking=True)
    torch.cuda.current_stream().synchronize()
    total = int(h_off[-1])
    h_out = torch.empty(total, dtype=torch.uint8, pin_memory=True)
    h_out.copy_(d_out[:total], non_blocking=True)
    ctx.stats()
    o, orec, _ = run_oracle(ev, *dims)
    assert 0 < total < orec.size                          # it is a compression
    dense = sparse_to_dense(bytes(h_out.numpy()), [int(v) for v in h_off.numpy()], S, P)
    assert dense.shape == orec.shape and (dense == orec).all()      # the reader restores the dense header too
    ctx.close()
