"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI binding and the oracle
on the same bytes, compare element by element."""
import numpy as np

from oracle import Oracle


def run_gpu(events, R, T, S, P, step_base, sorted_hint=True, cuts=None, path=None, grid=None, spill=0):
    """events: EVENT_DTYPE array (host).  Returns (records uint8 [R*T, rb], diag dict, (nv, ni), spans_out)."""
    import torch
    from paper_2606_20374_b200 import argus as A
    n_all = np.ascontiguousarray(events).nbytes // 32
    biggest = n_all if cuts is None else max([b - a for a, b in zip(cuts[:-1], cuts[1:])] + [0])
    grouped = path == 3 or (path is None and not sorted_hint)
    ctx = A.Argus(R, T, S, P, step_base, sorted_hint=sorted_hint,
                  max_ungrouped_events=biggest if grouped else 0, max_spill_events=spill)
    if path is not None:
        ctx.tune(A.TUNE_FORCE_PATH, path)
    if grid is not None:
        ctx.tune(A.TUNE_GRID_CTAS, grid)
    raw = np.ascontiguousarray(events).view(np.uint8).reshape(-1)
    d_ev = torch.from_numpy(raw.copy()).cuda() if raw.size else torch.empty(0, dtype=torch.uint8, device="cuda")
    rec = ctx.alloc_records()
    rec.fill_(0xAB)                      # garbage: the path must define every byte
    ctx.reset(rec)
    n = raw.size // 32
    cuts = [0, n] if cuts is None else cuts
    for a, b in zip(cuts[:-1], cuts[1:]):
        ctx.aggregate(d_ev.data_ptr() + a * 32 if b > a else None, b - a, rec)
    spans_out = torch.empty(R * T * (P + 1) * 32, dtype=torch.uint8, device="cuda")
    ctx.phase_times(rec, spans_out)
    outs = ctx.alloc_diag()
    for v in outs.values():
        v.fill_(0x5A if v.dtype == torch.uint8 else 0x5A5A5A5A)
    ctx.diagnose(rec, outs)
    stats = ctx.stats()
    out = (ctx.records_to_host(rec), ctx.diag_to_host(outs), stats,
           spans_out.cpu().numpy().view(A.SPAN_DTYPE).reshape(R, T, P + 1))
    ctx.close()
    return out


def run_oracle(events, R, T, S, P, step_base):
    o = Oracle(R, T, S, P, step_base)
    o.aggregate(events)
    return o, o.records(), o.diagnose()


def first_diff(a, b):
    d = np.nonzero(a.reshape(-1) != b.reshape(-1))[0]
    return None if d.size == 0 else int(d[0])


def compare_with_oracle(rec, diag, stats, spans_out, events, R, T, S, P, step_base):
    """Every record byte, the compact spans, the counters and the six diagnosis outputs against the oracle."""
    o, orec, odiag = run_oracle(events, R, T, S, P, step_base)
    assert stats == (o.n_valid, o.n_invalid)
    if not (rec == orec).all():
        i = first_diff(rec, orec)
        rb = rec.shape[1]
        raise AssertionError(f"records differ at byte {i}: record {i // rb} offset {i % rb} "
                             f"gpu={rec.reshape(-1)[i]} oracle={orec.reshape(-1)[i]} "
                             f"({int((rec != orec).sum())} bytes differ)")
    if spans_out is not None:
        assert (spans_out == o.spans()).all()
    for k in ("sig_stats", "sig_flags", "span_stats", "span_flags", "rank_score", "step_anomalous"):
        assert (diag[k] == odiag[k]).all(), (k, first_diff(diag[k].view(np.uint8), odiag[k].view(np.uint8)))
    return o


def assert_parity(events, R, T, S, P, step_base, **kw):
    rec, diag, stats, spans_out = run_gpu(events, R, T, S, P, step_base, **kw)
    o = compare_with_oracle(rec, diag, stats, spans_out, events, R, T, S, P, step_base)
    return rec, diag, o
