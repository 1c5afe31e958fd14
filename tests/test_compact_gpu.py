"""-m gpu parity tests of the compact record encodings (NEXT-4, second half; R37 sparse, R38 triple) through the
C ABI against oracle/compact.py: the byte streams and the offsets must be identical (integer / byte work:
bit-exact)."""
import dataclasses

import numpy as np
import pytest

from helpers import make_events, parse_compact_golden, parse_handworked
from oracle import Oracle
from oracle import compact as OC
from oracle import paper_literal as PL
from paper_2606_20374_b200.workload import build_workload, scaled

pytestmark = pytest.mark.gpu


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run(ev, R, T, S, P, base, capacity=None, **kw):
    """Aggregate + finalise on the GPU; returns (ctx, rec, oracle table)."""
    from paper_2606_20374_b200 import argus as A
    ctx = A.Argus(R, T, S, P, base, **kw)
    rec = ctx.alloc_records()
    ctx.reset(rec)
    if ev.size:
        ctx.aggregate(_cuda(ev.view(np.uint8).reshape(-1)), ev.size, rec)
    ctx.phase_times(rec)
    o = Oracle(R, T, S, P, base)
    o.aggregate(ev)
    o.phase_times()
    return ctx, rec, o


def _sparse(ctx, rec, n_rec, capacity=None):
    import torch
    cap = ctx.sparse_bound() if capacity is None else capacity
    out = torch.full((max(cap, 8),), 0xAB, dtype=torch.uint8, device="cuda")
    off = torch.zeros(n_rec + 1, dtype=torch.int64, device="cuda")
    ctx.sparse_encode(rec, out[:cap] if cap else out[:0], off)
    return out.cpu().numpy(), [int(v) for v in off.cpu().numpy()]


def test_sparse_handworked_bytes():
    g = parse_handworked()
    gold = parse_compact_golden()
    ctx, rec, o = _run(g["events"], 3, 1, 2, 2, 0)
    got, off = _sparse(ctx, rec, 3)
    assert off == [0, 240, 424, 656]
    for r in range(3):
        assert bytes(got[off[r]:off[r + 1]]) == bytes(gold["sparse"][r]), r
    ctx.close()


@pytest.mark.parametrize("name,kw", [
    ("tiny", dict(n_events=700)),                                     # many empty cells and phases
    ("tiny", dict()),
    ("mid", dict(n_ranks=5, n_steps=3, n_events=9000, n_sigs=517)),   # S not a multiple of the tile, ragged tail
    ("unsorted", dict(n_ranks=6, n_steps=2, n_events=4000, n_sigs=300)),   # heavy tail: wide bucket ranges
])
def test_sparse_stream_matches_oracle(name, kw):
    wl = build_workload(scaled(name, **kw))
    ev = wl.expand_host().copy()
    ev["end_ns"][::211] = -1                                        # invalid events: absent from both sides
    s = wl.spec
    ctx, rec, o = _run(ev, s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base,
                       sorted_hint=not s.shuffle, max_ungrouped_events=ev.size if s.shuffle else 0)
    want, woff = OC.sparse_encode(o.records(), s.n_sigs, s.n_phases)
    got, off = _sparse(ctx, rec, s.n_ranks * s.n_steps)
    assert off == woff
    assert bytes(got[:off[-1]]) == want
    assert off[-1] <= ctx.sparse_bound()
    ctx.close()


def test_sparse_edges_empty_table_top_bucket_and_short_buffer():
    # empty table: every record is header + mask
    ctx, rec, o = _run(make_events([]), 2, 2, 3, 2, 0)
    want, woff = OC.sparse_encode(o.records(), 3, 2)
    got, off = _sparse(ctx, rec, 4)
    assert off == woff == [0, 72, 144, 216, 288] and bytes(got[:288]) == want
    ctx.close()
    # a cell from bucket 0 to bucket 31 (nb = 32), and a buffer one byte short of the second record
    ev = make_events([(0, 0, 1, 0, 0, 10, 11), (0, 0, 1, 0, 1, 10, 10 + (1 << 40)), (1, 0, 0, 0, 0, 5, 9)])
    ctx, rec, o = _run(ev, 2, 1, 2, 2, 0)
    want, woff = OC.sparse_encode(o.records(), 2, 2)
    got, off = _sparse(ctx, rec, 2)
    assert off == woff and bytes(got[:off[-1]]) == want
    got, off = _sparse(ctx, rec, 2, capacity=woff[2] - 8)
    assert off == woff                                              # offsets complete: the caller sees it did not fit
    assert bytes(got[:woff[1]]) == want[:woff[1]]                   # the record that fits is written
    assert (got[woff[1]:woff[2] - 8] == 0xAB).all()                 # the one that does not is not touched
    ctx.close()


def test_triple_stream_matches_oracle():
    """events -> records -> 32-bucket KDE clusters (argus_kde_clusters_records) -> triple records, against the
    oracle chain on the oracle's own table (bimodal sigs: cells with one and with two clusters)."""
    import torch
    from paper_2606_20374_b200 import argus as A
    spec = dataclasses.replace(scaled("mid", n_ranks=4, n_steps=2, n_events=20_000, n_sigs=130), bimodal_frac=0.4)
    wl = build_workload(spec)
    ev = wl.expand_host()
    s = wl.spec
    R, T, S, P = s.n_ranks, s.n_steps, s.n_sigs, s.n_phases
    ctx, rec, o = _run(ev, R, T, S, P, s.step_base, max_spill_events=ev.size)
    MC = 4
    n_cells = R * T * S
    d_c = torch.zeros(n_cells * MC * 8, dtype=torch.uint8, device="cuda")
    d_n = torch.zeros(n_cells, dtype=torch.uint8, device="cuda")
    ctx.kde_clusters_records(rec, ctx.kde_params(per_octave=1, n_bins=32, max_clusters=MC), d_c, d_n)
    cap = ctx.triple_bound(MC)
    out = torch.full((cap,), 0xCD, dtype=torch.uint8, device="cuda")
    off = torch.zeros(R * T + 1, dtype=torch.int64, device="cuda")
    ctx.triple_encode(rec, d_c, d_n, MC, out, off)
    hist = o.cells()["hist"].reshape(R * T, S, 32)
    cl = [[PL.kde_clusters(hist[k, sg], per_octave=1, max_clusters=MC, min_gap_bins=0)[3] for sg in range(S)]
          for k in range(R * T)]
    assert max(len(c) for row in cl for c in row) >= 2
    want, woff = OC.triple_encode(o.records(), S, P, cl)
    assert [int(v) for v in off.cpu().numpy()] == woff
    assert bytes(out.cpu().numpy()[:woff[-1]]) == want
    # the handworked fixture's clusters, straight into the encoder
    ctx.close()
    g = parse_handworked()
    gold = parse_compact_golden()
    ctx, rec, o = _run(g["events"], 3, 1, 2, 2, 0)
    c = np.zeros((3, 2, 2), dtype=A.CLUSTER_DTYPE)
    n = np.zeros((3, 2), dtype=np.uint8)
    for (r, sg), tr in gold["clusters"].items():
        n[r, sg] = len(tr)
        for j, (cnt, p50, p99) in enumerate(tr):
            c[r, sg, j] = (cnt, p50, p99)
    out = torch.zeros(ctx.triple_bound(2), dtype=torch.uint8, device="cuda")
    off = torch.zeros(4, dtype=torch.int64, device="cuda")
    ctx.triple_encode(rec, _cuda(c.view(np.uint8).reshape(-1)), _cuda(n.reshape(-1)), 2, out, off)
    offs = [int(v) for v in off.cpu().numpy()]
    assert offs == [0, 176, 328, 496]
    got = out.cpu().numpy()
    for r in range(3):
        assert bytes(got[offs[r]:offs[r + 1]]) == bytes(gold["triple"][r]), r
    # a count beyond the slots of a cell is read as max_clusters (include/argus.h): same stream as the clamped input
    over = np.where(n == 2, 255, n).astype(np.uint8)
    assert (over > 2).any()
    out2 = torch.zeros_like(out)
    off2 = torch.zeros_like(off)
    ctx.triple_encode(rec, _cuda(c.view(np.uint8).reshape(-1)), _cuda(over.reshape(-1)), 2, out2, off2)
    assert [int(v) for v in off2.cpu().numpy()] == offs
    assert (out2.cpu().numpy()[:offs[-1]] == got[:offs[-1]]).all()
    ctx.close()


def test_compact_argument_errors():
    import torch
    from paper_2606_20374_b200 import argus as A
    ctx = A.Argus(2, 1, 4, 2)
    rec = ctx.alloc_records()
    ctx.reset(rec)
    out = torch.zeros(ctx.sparse_bound(), dtype=torch.uint8, device="cuda")
    off = torch.zeros(3, dtype=torch.int64, device="cuda")
    with pytest.raises(A.ArgusError) as e:
        ctx.sparse_encode(rec, out, off)                            # not finalised
    assert e.value.code == A.ESTATE
    ctx.phase_times(rec)
    with pytest.raises(A.ArgusError) as e:
        ctx.sparse_encode(rec, out[4:], off)                        # misaligned output
    assert e.value.code == A.EINVAL
    ctx.sparse_encode(rec, out, off)
    assert [int(v) for v in off.cpu().numpy()] == [0, 72, 144]
    ctx.close()
