"""Pins of oracle/compact.py (the R37 sparse and R38 triple record encodings), -m "not gpu": the hand-worked
byte fixture, an independent reader that must give back the dense table, the length formula, edge cases."""
import struct

import numpy as np

from helpers import make_events, parse_compact_golden, parse_handworked, sparse_to_dense
from oracle import Oracle
from oracle import compact as OC
from paper_2606_20374_b200.workload import build_workload, scaled


def _table(ev, R, T, S, P, base=0):
    o = Oracle(R, T, S, P, base)
    o.aggregate(ev)
    o.phase_times()
    return o.records()


def test_handworked_bytes():
    g = parse_handworked()
    gold = parse_compact_golden()
    rec = _table(g["events"], 3, 1, 2, 2)
    stream, off = OC.sparse_encode(rec, 2, 2)
    assert off == [0, 240, 424, 656]
    for r in range(3):
        assert stream[off[r]:off[r + 1]] == bytes(gold["sparse"][r]), r
    cl = [[gold["clusters"][(r, s)] for s in range(2)] for r in range(3)]
    stream, off = OC.triple_encode(rec, 2, 2, cl)
    assert off == [0, 176, 328, 496]
    for r in range(3):
        assert stream[off[r]:off[r + 1]] == bytes(gold["triple"][r]), r


def test_sparse_round_trip_tiny_and_length_formula():
    wl = build_workload(scaled("tiny", n_events=700))            # many empty cells, a few empty phases
    ev = wl.expand_host().copy()
    ev["start_ns"][::97] = -5                                      # invalid events are simply absent
    s = wl.spec
    rec = _table(ev, s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    stream, off = OC.sparse_encode(rec, s.n_sigs, s.n_phases)
    back = sparse_to_dense(stream, off, s.n_sigs, s.n_phases)
    assert np.array_equal(back, rec)
    # length = 64 + 8 + 32 * #non-empty phases + sum over non-empty cells (40 + 4 * (nb rounded up to even))
    o = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    o.aggregate(ev)
    cells, spans = o.cells().reshape(-1, s.n_sigs), o.spans().reshape(-1, s.n_phases + 1)
    for k in range(cells.shape[0]):
        want = 72 + 32 * int((spans[k, :s.n_phases]["n"] != 0).sum())
        for c in cells[k]:
            if c["count"]:
                nz = np.nonzero(c["hist"])[0]
                nb = int(nz[-1] - nz[0] + 1)
                want += 40 + 4 * (nb + (nb & 1))
        assert off[k + 1] - off[k] == want, k
    assert len(stream) < rec.size


def test_empty_table_and_top_bucket():
    rec = _table(make_events([]), 2, 2, 3, 2)
    stream, off = OC.sparse_encode(rec, 3, 2)
    assert off == [0, 72, 144, 216, 288]
    for k in range(4):
        assert struct.unpack_from("<Q", stream, off[k] + 64)[0] == 0          # no phase, no cell
        assert struct.unpack_from("<IQ", stream, off[k] + 20) [0] == 0
    assert np.array_equal(sparse_to_dense(stream, off, 3, 2), rec)
    # durations 1 ns and >= 2^31 ns in one cell: b0 = 0, nb = 32 (the widest entry, 40 + 128 bytes)
    ev = make_events([(0, 0, 1, 0, 0, 10, 11), (0, 0, 1, 0, 1, 10, 10 + (1 << 40))])
    rec = _table(ev, 1, 1, 2, 2)
    stream, off = OC.sparse_encode(rec, 2, 2)
    assert off[1] == 72 + 64 + 168
    assert struct.unpack_from("<IBBH", stream, 72 + 64) == (1, 0, 32, 0)
    assert np.array_equal(sparse_to_dense(stream, off, 2, 2), rec)


def test_triple_lengths():
    wl = build_workload(scaled("tiny", n_events=300))
    ev = wl.expand_host()
    s = wl.spec
    rec = _table(ev, s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    o = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    o.aggregate(ev)
    cells = o.cells().reshape(-1, s.n_sigs)
    cl = [[[(int(c["count"]), 3, 4)] * (1 + sg % 3) if c["count"] else [] for sg, c in enumerate(row)] for row in cells]
    stream, off = OC.triple_encode(rec, s.n_sigs, s.n_phases, cl)
    spans = o.spans().reshape(-1, s.n_phases + 1)
    for k in range(cells.shape[0]):
        want = 72 + 32 * int((spans[k, :s.n_phases]["n"] != 0).sum()) + sum(8 + 8 * len(t) for t in cl[k] if t)
        assert off[k + 1] - off[k] == want
        n_cells, = struct.unpack_from("<I", stream, off[k] + 20)
        assert n_cells == sum(1 for t in cl[k] if t)
