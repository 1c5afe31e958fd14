"""Pins of the CPU oracle (oracle/) against things other than itself: hand-worked golden values,
Python-int brute force, closed forms, invariants, fault recovery.  CPU only."""
import random

import numpy as np
import pytest

from helpers import (U64_MAX, check_against_bruteforce, check_handworked, make_events,
                     parse_handworked, parse_series_cases, py_bucket, py_series)
from oracle import Oracle, bucket, series
from paper_2606_20374_b200.workload import EVENT_DTYPE, build_workload, scaled


# ---- bucket (R4) ---------------------------------------------------------------------------
def test_bucket_powers_of_two():
    assert bucket(0) == 0 and bucket(1) == 0
    for k in range(64):
        for d in ((1 << k) - 1, 1 << k, (1 << k) + 1):
            if 0 <= d <= U64_MAX:
                assert bucket(d) == py_bucket(d), d
    assert bucket(U64_MAX) == 31
    # bucket b = [2^b, 2^(b+1)) for 1 <= b <= 30; bucket 31 is the clamp (>= 2.147 s)
    assert bucket(2**31 - 1) == 30 and bucket(2**31) == 31 and bucket(2**40) == 31
    assert bucket(2) == 1 and bucket(3) == 1 and bucket(4) == 2


def test_bucket_random():
    rnd = random.Random(1)
    for _ in range(2000):
        d = rnd.getrandbits(rnd.randint(1, 64))
        assert bucket(d) == py_bucket(d)


# ---- golden: the hand-worked example ---------------------------------------------------------
def test_handworked_example():
    g = parse_handworked()
    o = Oracle(3, 1, 2, 2, 0)
    o.aggregate(g["events"])
    check_handworked(g, o.cells(), o.spans(), o.n_valid, o.n_invalid, o.diagnose())


def test_series_closed_forms_golden():
    for x, med, mad, fl in parse_series_cases():
        m, d, nh, nl, flags = series(x)
        assert (m, d) == (med, mad), x
        assert list(flags) == fl, x
        assert (nh, nl) == (fl.count(1), fl.count(2))


# ---- brute force on tiny random inputs, including invalid records ----------------------------
def _random_events(rnd, n, R, T, S, P, step_base, big=False):
    rows = []
    for _ in range(n):
        r = rnd.randrange(R + (1 if rnd.random() < 0.02 else 0))
        st = step_base + rnd.randrange(-1 if rnd.random() < 0.02 else 0, T + (1 if rnd.random() < 0.02 else 0))
        s = rnd.randrange(S + (1 if rnd.random() < 0.02 else 0))
        ph = rnd.randrange(P + (1 if rnd.random() < 0.02 else 0))
        a = rnd.randrange(0, 10**9)
        if rnd.random() < 0.01:
            a = -rnd.randrange(1, 100)
        mode = rnd.random()
        if mode < 0.02:
            d = -rnd.randrange(1, 1000)          # end < start
        elif mode < 0.06:
            d = rnd.choice([0, 1, 2, 3])
        elif big and mode < 0.2:
            d = rnd.getrandbits(rnd.randint(30, 62))
        else:
            d = int(rnd.lognormvariate(10, 1.5))
        rows.append((r, max(st, 0), s, rnd.randrange(65536), ph, a, min(a + d, 2**63 - 1)))
    return make_events(rows)


@pytest.mark.parametrize("seed,dims,big", [(1, (3, 2, 5, 2, 0), False), (2, (8, 3, 16, 4, 10), True),
                                           (3, (1, 1, 1, 1, 0), True), (4, (5, 1, 7, 3, 1000), False)])
def test_aggregate_vs_python_bruteforce(seed, dims, big):
    R, T, S, P, base = dims
    rnd = random.Random(seed)
    ev = _random_events(rnd, 4000, R, T, S, P, base, big)
    o = Oracle(R, T, S, P, base)
    o.aggregate(ev)
    nv, ni = check_against_bruteforce(o.cells(), o.spans(), ev, R, T, S, P, base)
    assert (o.n_valid, o.n_invalid) == (nv, ni)
    assert ni > 0 and nv > 0


def test_sum_wraps_mod_2_64():
    # R6: two durations of 2^63 (needs start=0, end=2^63-1 max...) use 3 x (2^63-1) instead
    big = 2**63 - 1
    ev = make_events([(0, 0, 0, 0, 0, 0, big)] * 3)
    o = Oracle(1, 1, 1, 1, 0)
    o.aggregate(ev)
    c = o.cells()[0, 0, 0]
    assert int(c["sum"]) == (3 * big) % 2**64 and int(c["count"]) == 3
    assert int(c["hist"][31]) == 3


def test_empty_input_gives_identities():
    o = Oracle(2, 2, 3, 2, 0)
    o.aggregate(np.zeros(0, dtype=EVENT_DTYPE))
    c, s = o.cells(), o.spans()
    assert (c["count"] == 0).all() and (c["sum"] == 0).all() and (c["max"] == 0).all()
    assert (c["min"] == U64_MAX).all() and (c["hist"] == 0).all()
    assert (s["min_start"] == 2**63 - 1).all() and (s["max_end"] == -2**63).all()
    assert (s["span"] == 0).all() and (s["n"] == 0).all()
    d = o.diagnose()
    assert (d["sig_stats"]["median"] == 0).all() and (d["sig_flags"] == 0).all()
    assert (d["rank_score"] == 0).all() and (d["step_anomalous"] == 0).all()


# ---- median / MAD / flags vs Python sorted() -------------------------------------------------
@pytest.mark.parametrize("R", [1, 2, 3, 8, 9, 256, 257])
def test_series_vs_python_sorted(R):
    rnd = random.Random(R)
    for trial in range(30):
        kind = trial % 5
        if kind == 0:
            x = [rnd.getrandbits(64) for _ in range(R)]
        elif kind == 1:
            x = [rnd.randrange(5) for _ in range(R)]            # heavy ties
        elif kind == 2:
            x = [10**9 + int(rnd.gauss(0, 10**6)) for _ in range(R)]
            x[rnd.randrange(R)] *= 2
        elif kind == 3:
            x = [0] * R
            x[rnd.randrange(R)] = rnd.getrandbits(40)
        else:
            x = [rnd.getrandbits(rnd.randint(1, 64)) for _ in range(R)]
        med, mad, flags = py_series(x)
        m, d, nh, nl, fl = series(x)
        assert (m, d) == (med, mad)
        assert list(fl) == flags
        assert (nh, nl) == (flags.count(1), flags.count(2))


def test_series_translation_invariance():
    rnd = random.Random(5)
    for R in (4, 7, 64):
        x = [rnd.randrange(10**6) for _ in range(R)]
        m0, d0, _, _, f0 = series(x)
        c = 123456789
        m1, d1, _, _, f1 = series([v + c for v in x])
        assert m1 == m0 + c and d1 == d0 and list(f1) == list(f0)


def test_series_scaling_odd_R():
    # for odd R the median is an order statistic, so x -> c*x scales med and MAD exactly
    rnd = random.Random(6)
    for R in (3, 9, 101):
        x = [rnd.randrange(10**6) for _ in range(R)]
        m0, d0, _, _, f0 = series(x)
        m1, d1, _, _, f1 = series([7 * v for v in x])
        assert (m1, d1) == (7 * m0, 7 * d0) and list(f1) == list(f0)


# ---- invariants on generated workloads ------------------------------------------------------
def _agg(wl, ev=None):
    s = wl.spec
    ev = wl.expand_host() if ev is None else ev
    o = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    o.aggregate(ev)
    return o, ev


@pytest.fixture(scope="module")
def tiny():
    wl = build_workload("tiny")
    o, ev = _agg(wl)
    return wl, o, ev


def test_invariants_tiny(tiny):
    wl, o, ev = tiny
    s = wl.spec
    c, sp = o.cells(), o.spans()
    assert o.n_valid == s.total_events and o.n_invalid == 0
    assert (c["hist"].sum(axis=-1) == c["count"]).all()                     # buckets sum to count
    assert int(c["count"].sum()) == o.n_valid                               # counts sum to the total
    assert (c["count"].sum(axis=2) == sp["n"][:, :, s.n_phases]).all()
    ne = c["count"] > 0
    mean = c["sum"][ne] // c["count"][ne]
    assert (c["min"][ne] <= mean).all() and (mean <= c["max"][ne]).all()    # min <= sum/count <= max
    for cell in c[ne].reshape(-1)[:500]:
        nz = np.nonzero(cell["hist"])[0]
        assert py_bucket(int(cell["min"])) == nz[0] and py_bucket(int(cell["max"])) == nz[-1]
        lower = sum(int(cell["hist"][b]) * (0 if b == 0 else 1 << b) for b in range(32))
        upper = sum(int(cell["hist"][b]) * (1 << (b + 1)) for b in range(32))
        assert lower <= int(cell["sum"]) < upper
    # spans: whole = hull of the phases; span >= every phase span; sorted input -> first record
    P = s.n_phases
    assert (sp["min_start"][:, :, P] == sp["min_start"][:, :, :P].min(axis=2)).all()
    assert (sp["max_end"][:, :, P] == sp["max_end"][:, :, :P].max(axis=2)).all()
    assert (sp["span"][:, :, P:P + 1] >= sp["span"][:, :, :P]).all()
    first = ev.reshape(s.n_ranks, s.n_steps, s.n_events)[:, :, 0]
    assert (sp["min_start"][:, :, P] == first["start_ns"]).all()
    assert (sp["n"][:, :, :P].sum(axis=2) == sp["n"][:, :, P]).all()


def test_permutation_and_chunk_invariance(tiny):
    wl, o, ev = tiny
    s = wl.spec
    ref = o.records()
    rng = np.random.default_rng(7)
    o2 = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    o2.aggregate(ev[rng.permutation(ev.size)])
    assert (o2.records() == ref).all()
    o3 = Oracle(s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    cuts = [0, 1, 777, 2000, 2001, 31999, 50000, ev.size]      # cuts inside rank-steps (R7 merge)
    for a, b in zip(cuts[:-1], cuts[1:]):
        o3.aggregate(ev[a:b])
    assert (o3.records() == ref).all()


def test_record_layout(tiny):
    wl, o, ev = tiny
    s = wl.spec
    from oracle import CELL_DTYPE, HEADER_DTYPE, SPAN_DTYPE
    rec = o.records()
    assert rec.shape == (s.n_ranks * s.n_steps, 64 + 32 * (s.n_phases + 1) + 160 * s.n_sigs)
    hdr = rec[:, :64].copy().view(HEADER_DTYPE).reshape(-1)
    assert (hdr["magic"] == int.from_bytes(b"ARGS", "little")).all() and (hdr["version"] == 1).all()
    assert (hdr["n_sigs"] == s.n_sigs).all() and (hdr["n_phases"] == s.n_phases).all()
    assert list(hdr["rank"]) == [r for r in range(s.n_ranks) for _ in range(s.n_steps)]
    assert list(hdr["step"]) == [s.step_base + t for _ in range(s.n_ranks) for t in range(s.n_steps)]
    sp = rec[:, 64:64 + 32 * (s.n_phases + 1)].copy().view(SPAN_DTYPE)
    assert (sp.reshape(s.n_ranks, s.n_steps, -1) == o.spans()).all()
    ce = rec[:, 64 + 32 * (s.n_phases + 1):].copy().view(CELL_DTYPE)
    assert (ce.reshape(s.n_ranks, s.n_steps, -1) == o.cells()).all()
    assert (hdr["n_events"] == s.n_events).all()
    assert (hdr["iter_ns"] == o.spans()["span"][:, :, s.n_phases].reshape(-1)).all()
    # every header byte is pinned: the two timestamps against a Python-int brute force over the raw
    # events (first start / last end of each rank-step; swapping them in the oracle fails here), the
    # reserved words are zero, and nothing else lives in the 64 bytes
    assert (hdr["reserved0"] == 0).all() and (hdr["reserved1"] == 0).all()
    for i, h in enumerate(hdr):
        r, t = divmod(i, s.n_steps)
        sel = ev[(ev["rank"] == r) & (ev["step"] == s.step_base + t)]
        mn = min(int(v) for v in sel["start_ns"])
        mx = max(int(v) for v in sel["end_ns"])
        assert (int(h["min_start"]), int(h["max_end"]), int(h["iter_ns"])) == (mn, mx, mx - mn), (r, t)
        assert int(h["min_start"]) < int(h["max_end"])
    want = np.zeros(hdr.size, dtype=HEADER_DTYPE)
    for f in HEADER_DTYPE.names:
        want[f] = hdr[f]
    assert (want.view(np.uint8) == rec[:, :64].reshape(-1)).all()      # no byte outside the named fields


def test_record_header_handworked():
    """The H lines of tests/golden/handworked.txt (worked by hand) pin the oracle's header fields, and
    an untouched record's header carries the empty-span identities (R7, R17)."""
    from helpers import check_handworked_headers
    from oracle import HEADER_DTYPE
    g = parse_handworked()
    o = Oracle(3, 1, 2, 2, 0)
    o.aggregate(g["events"])
    rec = o.records()
    check_handworked_headers(g, rec[:, :64].copy().view(HEADER_DTYPE).reshape(3, 1))
    o2 = Oracle(2, 2, 3, 1, 50)
    o2.aggregate(make_events([(1, 51, 2, 0, 0, 10, 30)]))
    h = o2.records()[:, :64].copy().view(HEADER_DTYPE).reshape(2, 2)
    assert [int(h[1, 1][f]) for f in ("rank", "step", "n_events", "min_start", "max_end", "iter_ns")] == [1, 51, 1, 10, 30, 20]
    for r, t in ((0, 0), (0, 1), (1, 0)):
        assert [int(h[r, t][f]) for f in ("rank", "step", "n_events", "min_start", "max_end", "iter_ns")] == \
            [r, 50 + t, 0, 2**63 - 1, -2**63, 0]


# ---- detection: injected faults are recovered (recall only; precision is not asserted) --------
def test_tiny_faults_recovered(tiny):
    wl, o, ev = tiny
    d = o.diagnose()
    P = wl.spec.n_phases
    assert (d["sig_flags"][:, 17, 5] == 1).all()          # rank 5 is 1.5x slower on sig 17, all steps
    assert d["span_flags"][2, 1, 3] == 1                  # step 2: 2x-slow phase 1 on rank 3
    assert d["span_flags"][2, P, 3] == 1                  # ... visible in the iteration time too
    assert d["rank_score"][2].argmax() == 3


def test_mid_like_faults_recovered():
    wl = build_workload(scaled("mid", n_ranks=64, n_steps=2))
    o, ev = _agg(wl)
    d = o.diagnose()
    s = wl.spec
    counts = o.cells()["count"]
    from paper_2606_20374_b200.workload import sig_class
    score = d["rank_score"].sum(axis=0)
    bad = sorted(f.rank for f in wl.faults)
    assert sorted(np.argsort(score)[-len(bad):]) == bad    # stragglers are the top-K by rank_score
    for f in wl.faults:
        for t in range(s.n_steps):
            for sg in range(s.n_sigs):
                if sig_class(sg) == f.sig_class and counts[f.rank, t, sg] >= 16:
                    assert d["sig_flags"][t, sg, f.rank] == 1, (f, t, sg)


def test_unsorted_same_as_sorted():
    spec = scaled("unsorted", n_ranks=16, n_events=3000)
    wl = build_workload(spec)
    o, ev = _agg(wl)
    import dataclasses
    wl2 = build_workload(dataclasses.replace(spec, shuffle=False))
    o2, ev2 = _agg(wl2)
    key = lambda a: np.sort(a.view(np.dtype((np.void, 32))))
    assert (key(ev) == key(ev2)).all()                     # same multiset of records
    assert (o.records() == o2.records()).all()
    # heavy tail reaches far buckets
    assert np.nonzero(o.cells()["hist"].sum(axis=(0, 1, 2)))[0].max() >= 20


def test_rank_score_counts_high_only():
    # R = 5, S = 2.  sig 0: rank 4 ran it 10x longer (HIGH).  sig 1: rank 0 never ran it, its peers
    # did (x = 0 -> LOW, R11).  rank_score counts HIGH flags only (R14/R15).
    rows = [(r, 0, 0, 0, 0, 0, 1000 + r) for r in range(4)] + [(4, 0, 0, 0, 0, 0, 10000)]
    rows += [(r, 0, 1, 0, 0, 0, 500 + r) for r in range(1, 5)]
    o = Oracle(5, 1, 2, 1, 0)
    o.aggregate(make_events(rows))
    d = o.diagnose()
    assert list(d["sig_flags"][0, 0]) == [0, 0, 0, 0, 1]
    assert list(d["sig_flags"][0, 1]) == [2, 0, 0, 0, 0]
    assert list(d["rank_score"][0]) == [0, 0, 0, 0, 1]
    assert int(d["sig_stats"][0, 1]["n_low"]) == 1 and int(d["sig_stats"][0, 1]["n_high"]) == 0
