"""-m gpu parity tests: the CUDA path through the C ABI vs the CPU oracle, bit-exact (all work is
integer), on the same seeded bytes.  Sizes the oracle finishes in seconds, spanning several tiles
and ragged tails; the edge cases of DESIGN.md §3."""
import dataclasses
import random

import numpy as np
import pytest

from gpu_util import assert_parity, run_gpu
from helpers import check_handworked, make_events, parse_handworked, parse_series_cases
from paper_2606_20374_b200.workload import EVENT_DTYPE, build_workload, scaled

pytestmark = pytest.mark.gpu

PATH_SEG, PATH_GLOBAL, PATH_GROUPED = 1, 2, 3


def _dims(spec):
    return spec.n_ranks, spec.n_steps, spec.n_sigs, spec.n_phases, spec.step_base


def test_handworked_golden_gpu():
    from paper_2606_20374_b200 import argus as A
    g = parse_handworked()
    for path in (PATH_SEG, PATH_GLOBAL):
        rec, diag, stats, spans = run_gpu(g["events"], 3, 1, 2, 2, 0, path=path)
        ctx = A.Argus(3, 1, 2, 2, 0)
        hdr, sp, ce = ctx.split_records(rec)
        check_handworked(g, ce, sp, stats[0], stats[1], diag)
        assert (sp == spans).all()
        assert list(hdr["n_events"].reshape(-1)) == [3, 2, 2]
        assert list(hdr["iter_ns"].reshape(-1)) == [3148, 3200, 10000]
        ctx.close()


@pytest.mark.parametrize("path", [PATH_SEG, PATH_GLOBAL, PATH_GROUPED])
def test_tiny_parity(path):
    wl = build_workload("tiny")
    ev = wl.expand_host()
    rec, diag, o = assert_parity(ev, *_dims(wl.spec), path=path)
    assert (diag["sig_flags"][:, 17, 5] == 1).all() and diag["span_flags"][2, 1, 3] == 1


@pytest.mark.parametrize("path", [PATH_SEG, PATH_GLOBAL, PATH_GROUPED])
def test_tiny_chunked_mid_rank_step(path):
    wl = build_workload("tiny")
    ev = wl.expand_host()
    cuts = [0, 1, 777, 2000, 2001, 31999, 32000, 50000, ev.size]
    assert_parity(ev, *_dims(wl.spec), path=path, cuts=cuts)


def test_tiny_many_small_ctas():
    # rank-steps cut by CTA boundaries: the claim/merge protocol of the flush
    wl = build_workload("tiny")
    ev = wl.expand_host()
    for grid in (1, 3, 64, 1000):
        assert_parity(ev, *_dims(wl.spec), path=PATH_SEG, grid=grid)


def test_violated_sorted_hint_still_exact():
    wl = build_workload(scaled("tiny", n_ranks=4, n_steps=2, n_events=600))
    ev = wl.expand_host()
    rng = np.random.default_rng(3)
    assert_parity(ev[rng.permutation(ev.size)], *_dims(wl.spec), path=PATH_SEG)


def _random_events(rnd, n, R, T, S, P, base, big):
    rows = []
    for _ in range(n):
        r = rnd.randrange(R + (1 if rnd.random() < 0.02 else 0))
        st = base + rnd.randrange(-1 if (base and rnd.random() < 0.02) else 0, T + (1 if rnd.random() < 0.02 else 0))
        s = rnd.randrange(S + (1 if rnd.random() < 0.02 else 0))
        ph = rnd.randrange(P + (1 if rnd.random() < 0.02 else 0))
        a = rnd.randrange(0, 10**9)
        if rnd.random() < 0.01:
            a = -rnd.randrange(1, 100)
        mode = rnd.random()
        if mode < 0.02:
            d = -rnd.randrange(1, 1000)
        elif mode < 0.06:
            d = rnd.choice([0, 1, 2, 3])
        elif big and mode < 0.3:
            d = rnd.getrandbits(rnd.randint(1, 62))     # many buckets per sig, durations >= 2^32
        else:
            d = int(rnd.lognormvariate(10, 1.5))
        rows.append((r, st, s, rnd.randrange(65536), ph, a, min(a + d, 2**63 - 1)))
    rows.sort(key=lambda x: (x[0], x[1]))
    return make_events(rows)


@pytest.mark.parametrize("seed,dims,big", [(1, (3, 2, 5, 2, 0), False), (2, (8, 3, 16, 4, 10), True),
                                           (3, (1, 1, 1, 1, 0), True), (4, (5, 1, 7, 3, 1000), True),
                                           (5, (2, 2, 3, 64, 5), True)])
@pytest.mark.parametrize("path", [PATH_SEG, PATH_GLOBAL, PATH_GROUPED])
def test_random_with_invalid_and_overflow(seed, dims, big, path):
    R, T, S, P, base = dims
    ev = _random_events(random.Random(seed), 6000, R, T, S, P, base, big)
    rec, diag, o = assert_parity(ev, R, T, S, P, base, path=path)
    assert o.n_invalid > 0


@pytest.mark.parametrize("path", [PATH_SEG, PATH_GLOBAL, PATH_GROUPED])
def test_empty_input(path):
    ev = np.zeros(0, dtype=EVENT_DTYPE)
    assert_parity(ev, 4, 2, 9, 3, 0, path=path)


def test_sum_wrap_and_clamp_bucket():
    big = 2**63 - 1
    ev = make_events([(0, 0, 0, 0, 0, 0, big)] * 5 + [(1, 0, 1, 0, 0, 5, 5)])
    for path in (PATH_SEG, PATH_GLOBAL):
        assert_parity(ev, 2, 1, 2, 1, 0, path=path)


def test_hot_single_sig_carry():
    # one sig, one bucket, durations near 2^32: the u32 sum_lo carries constantly
    n = 50000
    ev = np.zeros(n, dtype=EVENT_DTYPE)
    ev["start_ns"] = np.arange(n)
    ev["end_ns"] = ev["start_ns"] + (2**32 - 1 - (np.arange(n) % 7))
    assert_parity(ev, 1, 1, 1, 1, 0, path=PATH_SEG)


def test_bucket_window_invariant_cells():
    # the compact cell holds at most four CONSECUTIVE buckets: sweep one sig over
    # every bucket upward, downward and bimodally (b and b+4 collide in the direct-mapped counters),
    # concurrently from all lanes, over several rank-steps; the refused events take the global path
    n_sig, R, T = 6, 3, 2
    rows = []
    t0 = 0
    for r in range(R):
        for t in range(T):
            for i in range(4000):
                k = i % 64
                up = (1 << (k % 33)) + (i % 3)                 # sig 0: all buckets upward (incl. >= 2^32)
                down = (1 << (32 - k % 33)) - (i % 2)          # sig 1: all buckets downward
                bi = (1 << 10) + i % 7 if i % 2 else (1 << 14) + i % 5   # sig 2: buckets 10 and 14
                tri = [3, 40, 700, 9000, 100000][i % 5]        # sig 3: five spread buckets
                edge = [(1 << 12) - 1, 1 << 12, (1 << 16) - 1, 1 << 16][i % 4]  # sig 4: window edges 11,12,15,16
                for s_, d in ((0, up), (1, down), (2, bi), (3, tri), (4, edge), (5, 1000 + i % 50)):
                    rows.append((r, t, s_, 0, i % 2, t0, t0 + d))
                    t0 += 7
    ev = make_events(rows)
    for grid in (None, 5):
        assert_parity(ev, R, T, n_sig, 2, 0, path=PATH_SEG, grid=grid)
        assert_parity(ev, R, T, n_sig, 2, 0, path=PATH_SEG, grid=grid, spill=ev.size)


@pytest.mark.parametrize("path", [PATH_SEG, PATH_GLOBAL])
def test_mid_scaled(path):
    wl = build_workload(scaled("mid", n_ranks=48, n_steps=3))
    ev = wl.expand_host()
    assert_parity(ev, *_dims(wl.spec), path=path)


def test_production_scaled_large_S():
    # S = 4096 (the compact table fills the CTA's shared memory), 16 phases, 8 streams, ragged N
    wl = build_workload(scaled("production", n_ranks=24, n_events=100_003))
    ev = wl.expand_host()
    assert_parity(ev, *_dims(wl.spec), path=PATH_SEG)


def test_unsorted_scaled():
    # shuffled input: without the hint the events are grouped first (path 3), then the segmented kernel
    wl = build_workload(scaled("unsorted", n_ranks=64, n_events=20000))
    ev = wl.expand_host()
    assert_parity(ev, *_dims(wl.spec), sorted_hint=False)
    assert_parity(ev, *_dims(wl.spec), sorted_hint=False, path=PATH_GLOBAL)
    # S <= 1024 runs three CTAs per SM with a short stage ring (5 stages of 8 KB; the geometry that once exposed a
    # stage released before its loads had landed): repeat, the race was timing dependent
    wl2 = build_workload(scaled("unsorted", n_ranks=64, n_events=20000, n_sigs=1000))
    ev2 = wl2.expand_host()
    for _ in range(3):
        assert_parity(ev2, *_dims(wl2.spec), sorted_hint=False)
    # the shuffled events in uneven chunks: every call groups its own chunk
    assert_parity(ev, *_dims(wl.spec), sorted_hint=False, cuts=[0, 7, 100_000, 100_001, 900_000, ev.size])


def test_multimodal_sigs_requeued():
    # same-name kernels "differ in duration by several multiples" between positions.  A share of
    # the sigs gets a second mode 8-4096x the first: the compact cell refuses it, the event is re-queued into
    # the CTA's spill region and folded at the flush of its rank-step; a third mode (or an exhausted region) falls
    # back to the overflow list.
    import dataclasses
    for name, kw, frac in (("mid", dict(n_ranks=24, n_steps=2), 0.5),
                           ("production", dict(n_ranks=8, n_events=150_001), 0.3),
                           ("unsorted", dict(n_ranks=16, n_events=20_000, shuffle=False), 0.0)):   # Pareto tails
        spec = dataclasses.replace(scaled(name, **kw), bimodal_frac=frac, bimodal_ratio=(8.0, 4096.0))
        wl = build_workload(spec)
        ev = wl.expand_host()
        for grid, spill in ((None, ev.size), (7, ev.size // 16), (None, 0), (3, 1000)):
            assert_parity(ev, *_dims(wl.spec), path=PATH_SEG, grid=grid, spill=spill)
    # the invariant sweep of test_bucket_window_invariant_cells (five spread buckets in one sig: a chain of
    # refusals in the replay) with a spill area, chunked
    wl = build_workload(dataclasses.replace(scaled("unsorted", n_ranks=32, n_events=6000), bimodal_frac=0.0))
    ev = wl.expand_host()
    assert_parity(ev, *_dims(wl.spec), sorted_hint=False, spill=ev.size, cuts=[0, 50_001, ev.size])


def test_odd_rank_counts_select():
    # R = 1, 2, 3, 9, 257, 4097 (odd/even medians, > 4096 ranks uses the 1024-thread select)
    rnd = random.Random(11)
    for R in (1, 2, 3, 9, 257, 4097):
        rows = []
        for r in range(R):
            for s in range(3):
                if rnd.random() < 0.9:
                    rows.append((r, 0, s, 0, s % 2, 1000 * r, 1000 * r + rnd.randrange(1, 10**6) * (50 if rnd.random() < 0.02 else 1)))
        assert_parity(make_events(rows), R, 1, 3, 2, 0, path=PATH_SEG)


def test_series_closed_forms_gpu():
    # golden series through the whole path: one event per rank with duration x (x < 2^63)
    for x, med, mad, fl in parse_series_cases():
        if max(x) >= 2**63:
            continue
        ev = make_events([(r, 0, 0, 0, 0, 0, v) for r, v in enumerate(x)])
        rec, diag, stats, _ = run_gpu(ev, len(x), 1, 1, 1, 0)
        st = diag["sig_stats"][0, 0]
        assert (int(st["median"]), int(st["mad"])) == (med, mad), x
        assert list(diag["sig_flags"][0, 0]) == fl, x


def test_device_expander_matches_host():
    import torch
    for name, kw in (("tiny", {}), ("mid", dict(n_ranks=8, n_steps=2)), ("unsorted", dict(n_ranks=8, n_events=3000))):
        wl = build_workload(scaled(name, **kw))
        h = wl.expand_host().view(np.uint8).reshape(-1)
        d = wl.expand_device().cpu().numpy()
        assert (h == d).all(), name


def test_grouping_with_many_groups():
    # R*T + 1 = 65,537 group counters do not fit shared memory: the grouping pass falls back to one
    # global counter array (L2 atomics); R*T = 32,768 uses the single scatter with per-CTA shared-memory
    # histograms; R*T = 3,000 the two-level grouping
    rnd = random.Random(5)
    for R, T in ((8192, 8), (16384, 2), (1000, 3)):
        rows = [(rnd.randrange(R + 1), 3 + rnd.randrange(T + 1), rnd.randrange(4), 0, rnd.randrange(2),
                 rnd.randrange(10**6), 10**6 + rnd.randrange(10**5)) for _ in range(30000)]
        assert_parity(make_events(rows), R, T, 4, 2, 3, sorted_hint=False)


def test_two_level_grouping_edges():
    """Ungrouped input through the two-level grouping pass: durations of 2^32 ns and more (they bypass the packed
    16-byte form), invalid events of every kind (dropped by the pass, re-appear as padding and must still be
    counted), a call of a few events, one whose events are all invalid, one whose events all bypass, a key
    count that is not a power of two, and several tiles per coarse bin."""
    rnd = random.Random(11)
    R, T, S, P, base = 37, 3, 50, 5, 1000
    rows = []
    for i in range(60_000):
        r, t, sg, ph = rnd.randrange(R), base + rnd.randrange(T), rnd.randrange(S), rnd.randrange(P)
        a = rnd.randrange(10**9)
        d = rnd.randrange(1, 10**5)
        k = rnd.random()
        if k < 0.02:
            d = (1 << 32) + rnd.randrange(1 << 33)              # bypasses the packed form
        elif k < 0.03:
            d = (1 << 32) - 1 - rnd.randrange(2)                # the largest packable durations
        elif k < 0.04:
            r = R + rnd.randrange(3)
        elif k < 0.05:
            t = base - 1 - rnd.randrange(2)
        elif k < 0.06:
            sg = S + rnd.randrange(100)
        elif k < 0.07:
            ph = P
        elif k < 0.08:
            a = -1 - rnd.randrange(100)
        elif k < 0.09:
            d = -1 - rnd.randrange(50)
        rows.append((r, t, sg, rnd.randrange(9), ph, a, a + d))
    ev = make_events(rows)
    assert_parity(ev, R, T, S, P, base, sorted_hint=False)
    assert_parity(ev, R, T, S, P, base, sorted_hint=False, cuts=[0, 3, 2051, 2052, 40_000, ev.size])
    bad = ev.copy()
    bad["sig"] = S + 1
    assert_parity(bad[:5000], R, T, S, P, base, sorted_hint=False)
    big = ev[(ev["end_ns"] - ev["start_ns"]) >= (1 << 32)]
    assert big.size > 500
    assert_parity(big, R, T, S, P, base, sorted_hint=False)
    one = ev.copy()                                              # every event in ONE key: a single coarse bin, 30 tiles
    one["rank"] = 7
    one["step"] = base + 1
    assert_parity(one, R, T, S, P, base, sorted_hint=False)
    assert_parity(ev[:1], R, T, S, P, base, sorted_hint=False)
