"""Shared test helpers: golden-file parsing and a pure-Python brute force (no numpy arithmetic on
the method's quantities: Python ints only) used to pin the C oracle."""
import os

import numpy as np

from paper_2606_20374_b200.workload import EVENT_DTYPE

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
U64_MAX = (1 << 64) - 1
I64_MAX = (1 << 63) - 1
I64_MIN = -(1 << 63)


def make_events(rows):
    """rows of (rank, step, sig, stream, phase, start, end) -> EVENT_DTYPE array."""
    ev = np.zeros(len(rows), dtype=EVENT_DTYPE)
    for i, r in enumerate(rows):
        ev[i] = tuple(r)
    return ev


def py_bucket(d: int) -> int:
    """R4 via int.bit_length (independent of the oracle's shift loop)."""
    return min(31, max(d.bit_length() - 1, 0))


def py_bruteforce(ev, R, T, S, P, step_base):
    """Dict-of-lists brute force of the first half: returns (cells, spans, n_valid, n_invalid)
    with cells[(r,t,s)] = list of durations, spans[(r,t,k)] = list of (start, end)."""
    cells, spans, nv, ni = {}, {}, 0, 0
    for e in ev:
        r, st, s, ph = int(e["rank"]), int(e["step"]), int(e["sig"]), int(e["phase"])
        a, b = int(e["start_ns"]), int(e["end_ns"])
        t = st - step_base
        if a < 0 or b < a or r >= R or t < 0 or t >= T or s >= S or ph >= P:
            ni += 1
            continue
        nv += 1
        cells.setdefault((r, t, s), []).append(b - a)
        spans.setdefault((r, t, ph), []).append((a, b))
        spans.setdefault((r, t, P), []).append((a, b))
    return cells, spans, nv, ni


def py_cell(durs):
    """Summary of a list of durations as Python ints (R5-R7)."""
    if not durs:
        return dict(count=0, sum=0, min=U64_MAX, max=0, hist=[0] * 32)
    h = [0] * 32
    for d in durs:
        h[py_bucket(d)] += 1
    return dict(count=len(durs), sum=sum(durs) & U64_MAX, min=min(durs), max=max(durs), hist=h)


def py_span(se):
    if not se:
        return dict(min_start=I64_MAX, max_end=I64_MIN, span=0, n=0)
    a = min(x[0] for x in se)
    b = max(x[1] for x in se)
    return dict(min_start=a, max_end=b, span=b - a, n=len(se))


def py_series(x):
    """NS rule with Python sorted() and ints: (median, mad, flags)."""
    R = len(x)
    v = sorted(x)
    lo, hi = v[(R - 1) // 2], v[R // 2]
    med = lo + (hi - lo) // 2
    dev = [abs(a - med) for a in x]
    w = sorted(dev)
    mad = w[(R - 1) // 2] + (w[R // 2] - w[(R - 1) // 2]) // 2
    thr = min(3 * mad, U64_MAX)
    flags = [(1 if a > med else 2) if d > thr else 0 for a, d in zip(x, dev)]
    return med, mad, flags


def check_against_bruteforce(cells_arr, spans_arr, ev, R, T, S, P, step_base):
    """cells_arr [R][T][S] CELL-like, spans_arr [R][T][P+1] SPAN-like structured arrays."""
    cells, spans, nv, ni = py_bruteforce(ev, R, T, S, P, step_base)
    for r in range(R):
        for t in range(T):
            for s in range(S):
                want = py_cell(cells.get((r, t, s), []))
                got = cells_arr[r, t, s]
                assert int(got["count"]) == want["count"], (r, t, s)
                assert int(got["sum"]) == want["sum"], (r, t, s)
                assert int(got["min"]) == want["min"], (r, t, s)
                assert int(got["max"]) == want["max"], (r, t, s)
                assert [int(v) for v in got["hist"]] == want["hist"], (r, t, s)
            for k in range(P + 1):
                want = py_span(spans.get((r, t, k), []))
                got = spans_arr[r, t, k]
                for f in ("min_start", "max_end", "span", "n"):
                    assert int(got[f]) == want[f], (r, t, k, f)
    return nv, ni


def parse_handworked():
    ev, cells, spans, ds, dp, hdrs = [], [], [], [], [], []
    n = rs = sa = None
    with open(os.path.join(GOLDEN, "handworked.txt")) as f:
        for line in f:
            p = line.split()
            if not p or p[0].startswith("#"):
                continue
            k, a = p[0], p[1:]
            if k == "E":
                ev.append(tuple(int(v) for v in a))
            elif k == "N":
                n = (int(a[0]), int(a[1]))
            elif k == "C":
                hist = [0] * 32
                for tok in a[6:]:
                    b, c = tok.split(":")
                    hist[int(b)] = int(c)
                cells.append((int(a[0]), int(a[1]), [int(v) for v in a[2:6]], hist))
            elif k == "S":
                spans.append((int(a[0]), int(a[1]), [int(v) for v in a[2:6]]))
            elif k == "H":
                hdrs.append(tuple(int(v) for v in a))
            elif k == "DS":
                ds.append((int(a[0]), int(a[1]), int(a[2]), [int(v) for v in a[3:]]))
            elif k == "DP":
                dp.append((int(a[0]), int(a[1]), int(a[2]), [int(v) for v in a[3:]]))
            elif k == "RS":
                rs = [int(v) for v in a]
            elif k == "SA":
                sa = [int(v) for v in a]
    return dict(events=make_events(ev), n=n, cells=cells, spans=spans, ds=ds, dp=dp, rs=rs, sa=sa,
                headers=hdrs)


def check_handworked_headers(g, hdr, n_sigs=2, n_phases=2):
    """hdr: HEADER-like structured array [R][T] of any implementation vs the golden H lines."""
    assert len(g["headers"]) == hdr.size
    for r, t, n, mn, mx, it in g["headers"]:
        h = hdr[r, t]
        assert int(h["magic"]) == int.from_bytes(b"ARGS", "little") and int(h["version"]) == 1
        assert (int(h["n_phases"]), int(h["n_sigs"])) == (n_phases, n_sigs)
        assert (int(h["rank"]), int(h["step"])) == (r, t)
        assert (int(h["n_events"]), int(h["min_start"]), int(h["max_end"]), int(h["iter_ns"])) == (n, mn, mx, it), (r, t)
        assert int(h["reserved0"]) == 0 and int(h["reserved1"]) == 0


def parse_series_cases():
    out = []
    with open(os.path.join(GOLDEN, "series_cases.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            x, st, fl = [seg.split() for seg in line.split("|")]
            out.append(([int(v) for v in x], int(st[0]), int(st[1]), [int(v) for v in fl]))
    return out


def check_handworked(g, cells_arr, spans_arr, n_valid, n_invalid, diag):
    """Compare any implementation's outputs with the hand-worked golden values."""
    assert (n_valid, n_invalid) == g["n"]
    for r, s, (cnt, sm, mn, mx), hist in g["cells"]:
        c = cells_arr[r, 0, s]
        assert (int(c["count"]), int(c["sum"]), int(c["min"]), int(c["max"])) == (cnt, sm, mn, mx)
        assert [int(v) for v in c["hist"]] == hist
    for r, k, vals in g["spans"]:
        sp = spans_arr[r, 0, k]
        assert [int(sp[f]) for f in ("min_start", "max_end", "span", "n")] == vals, (r, k)
    for s, med, mad, fl in g["ds"]:
        st = diag["sig_stats"][0, s]
        assert (int(st["median"]), int(st["mad"])) == (med, mad)
        assert list(diag["sig_flags"][0, s]) == fl
        assert (int(st["n_high"]), int(st["n_low"])) == (fl.count(1), fl.count(2))
    for k, med, mad, fl in g["dp"]:
        st = diag["span_stats"][0, k]
        assert (int(st["median"]), int(st["mad"])) == (med, mad)
        assert list(diag["span_flags"][0, k]) == fl
    assert list(diag["rank_score"][0]) == g["rs"]
    assert list(diag["step_anomalous"]) == g["sa"]


# ---- compact encodings (R37 sparse, R38 triple) -----------------------------------------------------
def parse_compact_golden():
    """tests/golden/compact_handworked.txt -> dict(sparse={rank: bytes}, triple={rank: bytes},
    clusters={(rank, sig): [(count, p50, p99)...]})."""
    import struct
    out = dict(sparse={}, triple={}, clusters={})
    cur = None
    with open(os.path.join(GOLDEN, "compact_handworked.txt")) as f:
        for line in f:
            p = line.split()
            if not p or p[0].startswith("#"):
                continue
            if p[0] in ("SPARSE", "TRIPLE"):
                cur = out[p[0].lower()].setdefault(int(p[1]), bytearray())
            elif p[0] == "CLUSTERS":
                v = [int(x) for x in p[3:]]
                out["clusters"][(int(p[1]), int(p[2]))] = [tuple(v[i:i + 3]) for i in range(0, len(v), 3)]
            else:
                cur += struct.pack("<" + p[0], *[int(x, 0) for x in p[1:]])
    return out


def sparse_to_dense(stream: bytes, offsets, S: int, P: int) -> np.ndarray:
    """An independent READER of the R37 sparse stream (walks it with an explicit cursor and rebuilds the dense
    R17 table, identities of R7 for what the stream leaves out) — used to pin the oracle's writer."""
    import struct
    rb = 64 + 32 * (P + 1) + 160 * S
    table = np.zeros((len(offsets) - 1, rb), dtype=np.uint8)
    for k in range(len(offsets) - 1):
        pos, end = offsets[k], offsets[k + 1]
        magic, ver, n_ph, n_sg, rank, step, n_cells, n_ev, mn, mx, it, length = struct.unpack_from("<IHHIIIIQqqQQ", stream, pos)
        assert (magic, ver, n_ph, n_sg, length) == (0x53475241, 2, P, S, end - pos)
        rec = bytearray(rb)
        struct.pack_into("<IHHIIIIQqqQQ", rec, 0, magic, 1, n_ph, n_sg, rank, step, 0, n_ev, mn, mx, it, 0)
        for j in range(P):
            struct.pack_into("<qqQQ", rec, 64 + 32 * j, I64_MAX, I64_MIN, 0, 0)
        struct.pack_into("<qqQQ", rec, 64 + 32 * P, mn, mx, it, n_ev)
        for s in range(S):
            struct.pack_into("<QQQQ", rec, 64 + 32 * (P + 1) + 160 * s, 0, 0, U64_MAX, 0)
        pos += 64
        mask, = struct.unpack_from("<Q", stream, pos)
        pos += 8
        for j in range(P):
            if mask >> j & 1:
                rec[64 + 32 * j: 96 + 32 * j] = stream[pos:pos + 32]
                pos += 32
        assert mask >> P == 0
        last = -1
        for _ in range(n_cells):
            s, b0, nb, z = struct.unpack_from("<IBBH", stream, pos)
            assert s > last and z == 0 and 1 <= nb and b0 + nb <= 32
            last = s
            c0 = 64 + 32 * (P + 1) + 160 * s
            rec[c0:c0 + 32] = stream[pos + 8: pos + 40]
            hist = struct.unpack_from("<%dI" % nb, stream, pos + 40)
            struct.pack_into("<%dI" % nb, rec, c0 + 32 + 4 * b0, *hist)
            pos += 40 + 4 * nb
            if nb & 1:
                assert struct.unpack_from("<I", stream, pos)[0] == 0
                pos += 4
        assert pos == end, (k, pos, end)
        table[k] = np.frombuffer(bytes(rec), dtype=np.uint8)
    return table
