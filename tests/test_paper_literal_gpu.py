"""-m gpu parity tests of the paper-literal float rows (SURVEY §8(f) NEXT-1..3) through the C ABI against
oracle/paper_literal.py on the same seeded inputs.
Tolerances: integers (bins, cluster counts, boundaries as cluster extents, flags, classes,
interval ends, widths, change-point steps) exact; fp64 quantities rel 1e-9 (the kernels and numpy sum in
different orders and call different exp / erfc / log implementations: a few ulp each over <= 4096 terms)."""
import math
import random

import numpy as np
import pytest

from helpers import make_events
from oracle import paper_literal as PL
from paper_2606_20374_b200.workload import build_workload, scaled

pytestmark = pytest.mark.gpu
RTOL = 1e-9


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _dims(spec):
    return spec.n_ranks, spec.n_steps, spec.n_sigs, spec.n_phases, spec.step_base


# ---- NEXT-1 -------------------------------------------------------------------------------------------
def test_fine_bin_thresholds_exhaustive():
    """Every bin threshold of R23 (floor(8 log2 d), decided in integers) from both sides, 0, 1, 2^32-1, >= 2^32,
    against the oracle's big-int rule, through argus_fine_hist."""
    import torch
    from paper_2606_20374_b200 import argus as A
    ds = {0, 1, 2, 3, 2**32 - 1, 2**32, 2**40, 2**62}
    for k in range(8, 256):
        lo, hi = 1, 1 << 33
        while lo < hi:
            mid = (lo + hi + 1) // 2
            if mid ** 8 < (1 << k):
                lo = mid
            else:
                hi = mid - 1
        ds.update((lo, lo + 1))
    rnd = random.Random(3)
    ds.update(rnd.getrandbits(rnd.randint(2, 34)) for _ in range(3000))
    ds = sorted(ds)
    # one event per sig: the sig tells which duration it was
    ev = make_events([(0, 0, i, 0, 0, 5, 5 + d) for i, d in enumerate(ds)])
    S = len(ds)
    ctx = A.Argus(1, 1, S, 1)
    hist = torch.zeros(S * 256, dtype=torch.int32, device="cuda")
    ctx.fine_hist(_cuda(ev.view(np.uint8).reshape(-1)), ev.size, hist)
    got = hist.cpu().numpy().reshape(S, 256)
    assert (got.sum(axis=1) == 1).all()
    assert [int(np.argmax(got[i])) for i in range(S)] == [PL.fine_bin(d) for d in ds]
    ctx.close()


def _compare_clusters(got_c, got_n, hists, per_octave, **kw):
    for i, h in enumerate(hists):
        f, bw, bounds, want = PL.kde_clusters(h, per_octave=per_octave, **kw)
        assert int(got_n[i]) == len(want), (i, got_n[i], want)
        for j, (cnt, p50, p99) in enumerate(want):
            g = got_c[i, j]
            assert (int(g["count"]), int(g["p50_bin"]), int(g["p99_bin"])) == (cnt, p50, p99), (i, j)
        assert (got_c[i, len(want):]["count"] == 0).all()


def test_kde_clusters_on_seeded_histograms():
    import torch
    from paper_2606_20374_b200 import argus as A
    rnd = np.random.default_rng(11)
    hists = []
    for i in range(400):
        kind = i % 5
        n = int(rnd.integers(1, 4000))
        if kind == 0:                                   # unimodal, as the named workloads (jitter sigma 0.1)
            x = rnd.normal(rnd.uniform(8, 28), rnd.uniform(0.02, 0.3), n)
        elif kind == 1:                                 # bimodal, 8-64x apart
            m = rnd.uniform(8, 22)
            x = np.concatenate([rnd.normal(m, 0.1, n), rnd.normal(m + rnd.uniform(3, 6), 0.1, max(1, n // int(rnd.integers(1, 6))))])
        elif kind == 2:                                 # three modes + a few strays
            m = rnd.uniform(6, 16)
            x = np.concatenate([rnd.normal(m, 0.08, n), rnd.normal(m + 4, 0.15, n // 2 + 1), rnd.normal(m + 9, 0.05, n // 3 + 1),
                                rnd.uniform(2, 30, 5)])
        elif kind == 3:                                 # heavy tail
            x = np.log2(5000.0 * (1.0 - rnd.random(n)) ** (-1 / 1.5))
        else:                                           # nearly empty / single bin
            x = np.full(int(rnd.integers(0, 4)), rnd.uniform(5, 25))
        h = np.zeros(256, dtype=np.uint32)
        for v in x:
            h[PL.fine_bin(int(round(2.0 ** min(max(v, 0.0), 40.0))))] += 1
        hists.append(h)
    H = np.stack(hists)
    ctx = A.Argus(1, 1, 1, 1)
    for mc in (8, 2):
        p = ctx.kde_params(max_clusters=mc)
        d_c = torch.zeros(len(hists) * mc * 8, dtype=torch.uint8, device="cuda")
        d_n = torch.zeros(len(hists), dtype=torch.uint8, device="cuda")
        d_f = torch.zeros(len(hists) * 256, dtype=torch.float64, device="cuda")
        ctx.kde_clusters(_cuda(H), len(hists), p, d_c, d_n, d_f)
        got_c = d_c.cpu().numpy().view(A.CLUSTER_DTYPE).reshape(len(hists), mc)
        _compare_clusters(got_c, d_n.cpu().numpy(), hists, 8, max_clusters=mc)
        got_f = d_f.cpu().numpy().reshape(len(hists), 256)
        for i, h in enumerate(hists):
            f = PL.kde_clusters(h)[0]
            assert np.allclose(got_f[i], f, rtol=RTOL, atol=1e-13 * max(1e-300, f.max())), i   # far tails underflow differently
        # without the density the kernel gives eight lanes to a histogram whose occupied bins span <= 64 grid steps and
        # a warp to the wider ones (the strays of kind 2, the heavy tails): the same clusters either way
        spans = [int(np.nonzero(h)[0][-1] - np.nonzero(h)[0][0]) if h.any() else 0 for h in hists]
        assert min(spans) < 64 <= max(spans)
        d_c2 = torch.full((len(hists) * mc * 8,), 0xAB, dtype=torch.uint8, device="cuda")
        d_n2 = torch.full((len(hists),), 0xAB, dtype=torch.uint8, device="cuda")
        ctx.kde_clusters(_cuda(H), len(hists), p, d_c2, d_n2, None)
        assert torch.equal(d_n2, d_n) and torch.equal(d_c2, d_c)
        _compare_clusters(d_c2.cpu().numpy().view(A.CLUSTER_DTYPE).reshape(len(hists), mc), d_n2.cpu().numpy(), hists, 8,
                          max_clusters=mc)
    ctx.close()


def test_compression_from_records_and_from_fine_histograms():
    """The whole NEXT-1 path on a bimodal workload: events -> (a) the 32-bucket histograms of the records,
    (b) the 256-bin fine histograms -> clusters, both against the oracle run on the oracle's own histograms."""
    import dataclasses
    import torch
    from oracle import Oracle
    from paper_2606_20374_b200 import argus as A
    spec = dataclasses.replace(scaled("mid", n_ranks=6, n_steps=2, n_events=30_000, n_sigs=96), bimodal_frac=0.4)
    wl = build_workload(spec)
    ev = wl.expand_host()
    R, T, S, P, base = _dims(wl.spec)
    d_ev = _cuda(ev.view(np.uint8).reshape(-1))
    ctx = A.Argus(R, T, S, P, base, max_spill_events=ev.size)
    rec = ctx.alloc_records()
    ctx.reset(rec)
    ctx.aggregate(d_ev, ev.size, rec)
    ctx.phase_times(rec)
    n_cells = R * T * S
    # (a) coarse grid, straight from the record table
    p1 = ctx.kde_params(per_octave=1, n_bins=32, max_clusters=4)
    c1 = torch.zeros(n_cells * 4 * 8, dtype=torch.uint8, device="cuda")
    n1 = torch.zeros(n_cells, dtype=torch.uint8, device="cuda")
    ctx.kde_clusters_records(rec, p1, c1, n1)
    o = Oracle(R, T, S, P, base)
    o.aggregate(ev)
    coarse = o.cells()["hist"].reshape(n_cells, 32)
    _compare_clusters(c1.cpu().numpy().view(A.CLUSTER_DTYPE).reshape(n_cells, 4), n1.cpu().numpy(), coarse, 1,
                      max_clusters=4, min_gap_bins=0)
    # (b) fine grid
    hist = torch.zeros(n_cells * 256, dtype=torch.int32, device="cuda")
    ctx.fine_hist(d_ev, ev.size, hist)
    want_h = PL.fine_histograms(ev, R, T, S, P, base).reshape(n_cells, 256)
    assert np.array_equal(hist.cpu().numpy().view(np.uint32).reshape(n_cells, 256), want_h)
    p8 = ctx.kde_params(max_clusters=4)
    c8 = torch.zeros(n_cells * 4 * 8, dtype=torch.uint8, device="cuda")
    n8 = torch.zeros(n_cells, dtype=torch.uint8, device="cuda")
    ctx.kde_clusters(hist, n_cells, p8, c8, n8)
    got_n = n8.cpu().numpy()
    _compare_clusters(c8.cpu().numpy().view(A.CLUSTER_DTYPE).reshape(n_cells, 4), got_n, want_h, 8, max_clusters=4)
    # the bimodal sigs come out as two clusters where they have enough samples, the others as one
    m2 = wl.tables["mode2_q16"]
    cnt = o.cells()["count"].reshape(R * T, S)
    two = got_n.reshape(R * T, S)
    assert (two[:, m2 == 0][cnt[:, m2 == 0] >= 32] == 1).mean() > 0.97
    assert (two[:, m2 != 0][cnt[:, m2 != 0] >= 200] == 2).mean() > 0.9
    ctx.close()


# ---- NEXT-2 -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("R,C,K,G", [(24, 2, 5, 128), (257, 3, 4, 64), (1, 1, 2, 16), (2, 2, 3, 32)])
def test_l3_scores_and_fence(R, C, K, G):
    import torch
    from paper_2606_20374_b200 import argus as A
    rnd = random.Random(100 + R)
    cnt = np.zeros((K, R, C), dtype=np.uint32)
    p50 = np.ones((K, R, C), dtype=np.float64)
    p99 = np.ones((K, R, C), dtype=np.float64)
    for k in range(K):
        base = [rnd.uniform(1e3, 1e7) * (30 ** c) for c in range(C)]
        for r in range(R):
            for c in range(C):
                if rnd.random() < 0.9:
                    slow = 1.6 if (r == k % R and R > 4) else 1.0
                    cnt[k, r, c] = rnd.randrange(1, 5000)
                    p50[k, r, c] = base[c] * slow * (1 + 0.02 * rnd.random())
                    p99[k, r, c] = p50[k, r, c] * (1.0 if rnd.random() < 0.1 else 1 + 0.6 * rnd.random())
    if K > 1:
        cnt[K - 1] = 0                                    # a key nobody ran
    ctx = A.Argus(1, 1, 1, 1)
    d_score = torch.zeros(K * R, dtype=torch.float64, device="cuda")
    d_stat = torch.zeros(K * 5, dtype=torch.float64, device="cuda")
    d_flags = torch.full((K * R,), 7, dtype=torch.uint8, device="cuda")
    ctx.l3_detect(_cuda(cnt), _cuda(p50), _cuda(p99), K, R, C, d_score, d_stat, d_flags, n_grid=G, alpha=1.5)
    score = d_score.cpu().numpy().reshape(K, R)
    stat = d_stat.cpu().numpy().view(A.L3_STAT_DTYPE).reshape(K)
    flags = d_flags.cpu().numpy().reshape(K, R)
    for k in range(K):
        tr = [[(int(cnt[k, r, c]), float(p50[k, r, c]), float(p99[k, r, c])) for c in range(C)] for r in range(R)]
        xs, F, W, want, q1, q3, fence, wflags = PL.l3_scores(tr, n_grid=G, alpha=1.5)
        scale = max(1e-300, float(np.abs(want).max()))
        assert np.allclose(score[k], want, rtol=1e-8, atol=1e-9 * scale), k
        assert stat[k]["q1"] == pytest.approx(q1, rel=1e-8, abs=1e-9 * scale)
        assert stat[k]["fence"] == pytest.approx(fence, rel=1e-8, abs=1e-9 * scale)
        if want.any():
            assert stat[k]["x_lo"] == pytest.approx(xs[0], rel=1e-12) and stat[k]["x_hi"] == pytest.approx(xs[-1], rel=1e-12)
        # flags: equal wherever the score is not within rounding of the fence
        clear = np.abs(want - fence) > 1e-7 * scale
        assert (flags[k][clear] == wflags[clear]).all(), k
        if want.any():
            assert int(np.argmax(score[k])) == int(np.argmax(want))      # the same rank deviates most
    ctx.close()


@pytest.mark.parametrize("R,C,G,quantised", [(4096, 2, 24, False), (1500, 3, 16, False), (1024, 1, 16, False),
                                             (4096, 1, 24, True), (3000, 2, 16, True)])
def test_l3_large_rank_counts_sampled(R, C, G, quantised):
    """The launch shapes of the full-size job (1,024 threads, 2 or 4 sorted positions per thread, every cached /
    uncached parameter path): the oracle's R x R matrix is out of reach, so the scores of SAMPLED ranks are
    compared with the oracle's own mixture_cdf / w1 summed over all the other ranks, the quartiles and the fence
    with numpy's percentile of the kernel's scores (R33's definition), the flags with score > fence.
    quantised: p50 / p99 take a few bin values and the counts a few values, as the triples of NEXT-1 do — most ranks
    then carry identical mixtures and the kernel scores the distinct ones with their multiplicities instead of
    sorting R values per grid point; the random cases have R distinct mixtures and take the sort."""
    import torch
    from paper_2606_20374_b200 import argus as A
    rnd = np.random.default_rng(7 + R)
    K = 2
    cnt = np.zeros((K, R, C), dtype=np.uint32)
    p50 = np.ones((K, R, C), dtype=np.float64)
    p99 = np.ones((K, R, C), dtype=np.float64)
    for k in range(K):
        base = 5e4 * (25.0 ** np.arange(C))
        have = rnd.random((R, C)) < (0.95 if k == 0 else 0.6)          # key 1: many ranks lack a cluster
        cnt[k] = np.where(have, rnd.integers(1, 4000, (R, C)), 0)
        p50[k] = base * (1 + 0.03 * rnd.random((R, C)))
        p99[k] = p50[k] * np.where(rnd.random((R, C)) < 0.15, 1.0, 1 + 0.5 * rnd.random((R, C)))
        if quantised:
            b50 = rnd.integers(0, 3, (R, C)) + (rnd.random((R, C)) < 0.01) * 5
            p50[k] = base * 2.0 ** ((b50 + 0.5) / 8.0)
            p99[k] = p50[k] * 2.0 ** (rnd.integers(0, 2, (R, C)) / 8.0)
            cnt[k] = np.where(have, rnd.choice([100, 200], (R, C)), 0)
        p50[k, 17] *= 1.7; p99[k, 17] *= 1.7                           # one rank is slow on every cluster
        cnt[k, 17] = np.maximum(cnt[k, 17], 1)
        cnt[k, 33] = 0                                                 # one rank never ran the kernel
    ctx = A.Argus(1, 1, 1, 1)
    d_score = torch.zeros(K * R, dtype=torch.float64, device="cuda")
    d_stat = torch.zeros(K * 5, dtype=torch.float64, device="cuda")
    d_flags = torch.full((K * R,), 7, dtype=torch.uint8, device="cuda")
    ctx.l3_detect(_cuda(cnt), _cuda(p50), _cuda(p99), K, R, C, d_score, d_stat, d_flags, n_grid=G, alpha=1.5)
    score = d_score.cpu().numpy().reshape(K, R)
    stat = d_stat.cpu().numpy().view(A.L3_STAT_DTYPE).reshape(K)
    flags = d_flags.cpu().numpy().reshape(K, R)
    for k in range(K):
        tr = [[(int(cnt[k, r, c]), float(p50[k, r, c]), float(p99[k, r, c])) for c in range(C)] for r in range(R)]
        live = [(t[1], t[2]) for row in tr for t in row if t[0] > 0]
        xs = PL.log_grid(0.5 * min(a for a, _ in live), 2.0 * max(b for _, b in live), G)
        assert stat[k]["x_lo"] == pytest.approx(xs[0], rel=1e-12) and stat[k]["x_hi"] == pytest.approx(xs[-1], rel=1e-12)
        F = np.stack([PL.mixture_cdf(row, xs) for row in tr])
        scale = float(score[k].max())
        for r in [0, 1, 17, 33, R // 2, R - 1] + [int(v) for v in rnd.integers(0, R, 10)]:
            want = sum(PL.w1(F[r], F[b], xs) for b in range(R) if b != r) / (R - 1)
            assert score[k, r] == pytest.approx(want, rel=1e-8, abs=1e-9 * scale), (k, r)
        q1, q3 = np.percentile(score[k], [25.0, 75.0])
        assert stat[k]["q1"] == pytest.approx(q1, rel=1e-12) and stat[k]["q3"] == pytest.approx(q3, rel=1e-12)
        fence = q3 + 1.5 * (q3 - q1)
        assert stat[k]["fence"] == pytest.approx(fence, rel=1e-12)
        assert (flags[k] == (score[k] > stat[k]["fence"])).all()
        assert np.isfinite(score[k]).all() and (score[k] >= 0).all()
    ctx.close()


def test_events_to_l3_end_to_end():
    """The paper's whole L3 route on one table (PAPER.md:176-198 then 234-251): events -> fine histograms ->
    clusters (argus_kde_clusters) -> regrouped triples in ns (argus_clusters_to_l3) -> scores, fence, flags
    (argus_l3_detect), against the oracle chained the same way on the oracle's own histograms.  tiny's
    injected fault (rank 5 x1.5 on sig 17) must carry the top score of its key in every step."""
    import torch
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("tiny", n_events=6000))
    ev = wl.expand_host()
    R, T, S, P, base = _dims(wl.spec)
    MC, G = 4, 64
    ctx = A.Argus(R, T, S, P, base)
    n_cells = R * T * S
    hist = torch.zeros(n_cells * 256, dtype=torch.int32, device="cuda")
    ctx.fine_hist(_cuda(ev.view(np.uint8).reshape(-1)), ev.size, hist)
    d_c = torch.zeros(n_cells * MC * 8, dtype=torch.uint8, device="cuda")
    d_n = torch.zeros(n_cells, dtype=torch.uint8, device="cuda")
    ctx.kde_clusters(hist, n_cells, ctx.kde_params(max_clusters=MC), d_c, d_n)
    K = T * S
    d_cnt = torch.full((K * R * MC,), 9, dtype=torch.int32, device="cuda")
    d_p50 = torch.zeros(K * R * MC, dtype=torch.float64, device="cuda")
    d_p99 = torch.zeros(K * R * MC, dtype=torch.float64, device="cuda")
    ctx.clusters_to_l3(d_c, MC, 8, d_cnt, d_p50, d_p99)
    d_score = torch.zeros(K * R, dtype=torch.float64, device="cuda")
    d_stat = torch.zeros(K * 5, dtype=torch.float64, device="cuda")
    d_flags = torch.zeros(K * R, dtype=torch.uint8, device="cuda")
    ctx.l3_detect(d_cnt, d_p50, d_p99, K, R, MC, d_score, d_stat, d_flags, n_grid=G, alpha=1.5)
    cnt = d_cnt.cpu().numpy().view(np.uint32).reshape(K, R, MC)
    p50 = d_p50.cpu().numpy().reshape(K, R, MC)
    p99 = d_p99.cpu().numpy().reshape(K, R, MC)
    score = d_score.cpu().numpy().reshape(K, R)
    flags = d_flags.cpu().numpy().reshape(K, R)
    stat = d_stat.cpu().numpy().view(A.L3_STAT_DTYPE).reshape(K)
    H = PL.fine_histograms(ev, R, T, S, P, base)
    for t in range(T):
        for s in range(S):
            k = t * S + s
            tr = []
            for r in range(R):
                cl = PL.kde_clusters(H[r, t, s], max_clusters=MC)[3]
                tr.append([(c, PL.bin_value_ns(b50), PL.bin_value_ns(b99)) for c, b50, b99 in cl])
                for j in range(MC):                       # the regrouped triples themselves
                    if j < len(cl):
                        assert int(cnt[k, r, j]) == cl[j][0]
                        assert p50[k, r, j] == pytest.approx(tr[r][j][1], rel=1e-14)
                        assert p99[k, r, j] == pytest.approx(tr[r][j][2], rel=1e-14)
                    else:
                        assert int(cnt[k, r, j]) == 0
            xs, F, W, want, q1, q3, fence, wflags = PL.l3_scores(tr, n_grid=G, alpha=1.5)
            # ranks with identical triples score exactly 0 on both sides (the kernel sums gaps of the sorted
            # CDF values times integers: no cancellation)
            scale = max(1e-300, float(np.abs(want).max()))
            assert np.allclose(score[k], want, rtol=1e-8, atol=1e-9 * scale), k
            assert stat[k]["fence"] == pytest.approx(fence, rel=1e-8, abs=1e-9 * scale)
            clear = np.abs(want - fence) > 1e-7 * scale
            assert (flags[k][clear] == wflags[clear]).all(), k
    for t in range(T):
        assert int(np.argmax(score[t * S + 17])) == 5 and flags[t * S + 17, 5] == 1
    ctx.close()


# ---- NEXT-3 -------------------------------------------------------------------------------------------
def test_l2_groups_on_a_table():
    import torch
    from oracle import Oracle
    from paper_2606_20374_b200 import argus as A
    wl = build_workload(scaled("mid", n_ranks=48, n_steps=3, n_events=3000))
    ev = wl.expand_host()
    R, T, S, P, base = _dims(wl.spec)
    ctx = A.Argus(R, T, S, P, base)
    rec = ctx.alloc_records()
    ctx.reset(rec)
    ctx.aggregate(_cuda(ev.view(np.uint8).reshape(-1)), ev.size, rec)
    ctx.phase_times(rec)
    # Table 3 routing: two dimensions; "DP groups" of 8 consecutive ranks, "EP groups" by rank mod 6 (one rank
    # outside every EP group, one group of a single rank)
    gid = np.zeros((2, R), dtype=np.uint32)
    gid[0] = np.arange(R) // 8
    gid[1] = np.arange(R) % 6
    gid[1, 7] = 0xFFFFFFFF
    gid[1, 9] = 40
    route = np.array([k % 2 for k in range(P + 1)], dtype=np.uint8)
    d_g = torch.zeros((P + 1) * R * 32, dtype=torch.uint8, device="cuda")
    d_z = torch.zeros((P + 1) * R, dtype=torch.float64, device="cuda")
    d_f = torch.zeros((P + 1) * R, dtype=torch.uint8, device="cuda")
    d_x = torch.zeros((P + 1) * R, dtype=torch.float64, device="cuda")
    ctx.l2_groups(rec, _cuda(route), _cuda(gid), 1.5, d_g, d_z, d_f, d_x)
    G = d_g.cpu().numpy().view(A.L2_GROUP_DTYPE).reshape(P + 1, R)
    z = d_z.cpu().numpy().reshape(P + 1, R)
    fl = d_f.cpu().numpy().reshape(P + 1, R)
    o = Oracle(R, T, S, P, base)
    o.aggregate(ev)
    span = o.spans()["span"].astype(np.float64)          # [R][T][P+1]
    for k in range(P + 1):
        xbar = span[:, :, k].sum(axis=1) / T
        g = gid[route[k]].astype(np.int64)
        member = g < R
        want, wz, wf = PL.l2_groups(xbar[member], g[member], z_thr=1.5)
        assert np.allclose(d_x.cpu().numpy().reshape(P + 1, R)[k], xbar, rtol=1e-15)
        for grp, (n, mu, sigma, cv, cls) in want.items():
            q = G[k, grp]
            assert int(q["n"]) == n and int(q["cls"]) == cls
            assert q["mu"] == pytest.approx(mu, rel=RTOL) and q["sigma"] == pytest.approx(sigma, rel=RTOL, abs=1e-9)
            assert q["cv"] == pytest.approx(cv, rel=RTOL, abs=1e-15)
        assert int((G[k]["n"] > 0).sum()) == len(want)
        assert np.allclose(z[k][member], wz, rtol=1e-8, atol=1e-9) and (z[k][~member] == 0).all()
        clear = np.abs(wz - 1.5) > 1e-6
        assert (fl[k][member][clear] == wf[clear]).all() and (fl[k][~member] == 0).all()
    # Fixed-order group sums: a second run gives the same BITS (the kernel has no floating-point atomics); and a
    # route byte beyond n_dims sends its event to no group instead of reading past d_group_id.
    route2 = route.copy()
    route2[0] = 7
    d_g2, d_z2, d_f2 = torch.full_like(d_g, 0x5A), torch.full_like(d_z, 3.0), torch.full_like(d_f, 9)
    ctx.l2_groups(rec, _cuda(route2), _cuda(gid), 1.5, d_g2, d_z2, d_f2, d_x)
    ctx.stats()
    G2 = d_g2.cpu().numpy().view(A.L2_GROUP_DTYPE).reshape(P + 1, R)
    assert (G2[1:].view(np.uint8) == G[1:].view(np.uint8)).all()
    assert (d_z2.cpu().numpy().reshape(P + 1, R)[1:].view(np.uint64) == z[1:].view(np.uint64)).all()
    assert (d_f2.cpu().numpy().reshape(P + 1, R)[1:] == fl[1:]).all()
    assert (G2[0]["n"] == 0).all() and (d_z2.cpu().numpy()[:R] == 0).all() and (d_f2.cpu().numpy()[:R] == 0).all()
    with pytest.raises(A.ArgusError) as e:
        ctx.l2_groups(rec, _cuda(route), _cuda(gid), 1.5, d_g, d_z, d_f, d_x, n_dims=0)
    assert e.value.code == A.EINVAL
    ctx.close()


def test_l1_jitter_and_change_point():
    import torch
    from paper_2606_20374_b200 import argus as A
    rnd = np.random.default_rng(5)
    T, n = 96, 40
    x = np.rint(1e8 * (1 + 0.004 * rnd.standard_normal((n, T)))).astype(np.uint64)
    for s in range(n):
        kind = s % 5
        if kind == 1:                                    # narrow spike(s)
            for _ in range(1 + s % 3):
                t = int(rnd.integers(0, T - 3))
                x[s, t:t + 1 + s % 4] = (x[s, t:t + 1 + s % 4] * 1.9).astype(np.uint64)
        elif kind == 2:                                  # step regression
            t = int(rnd.integers(10, T - 10))
            x[s, t:] = (x[s, t:] * 1.25).astype(np.uint64)
        elif kind == 3:                                  # both
            t = int(rnd.integers(20, T - 20))
            x[s, t:] = (x[s, t:] * 1.3).astype(np.uint64)
            x[s, 5] = x[s, 5] * 3
        elif kind == 4:                                  # noisy: no stable sides
            x[s] = np.rint(1e8 * (1 + 0.2 * rnd.random(T))).astype(np.uint64)
    ctx = A.Argus(1, 1, 1, 1)
    # the series live with a stride, as the whole-iteration span_ns inside argus_phase_times' d_spans_out
    P1 = 3
    buf = np.zeros((n, T, P1, 4), dtype=np.uint64)
    buf[:, :, P1 - 1, 2] = x
    d_buf = _cuda(buf)
    d_out = torch.zeros(n * A.L1_OUT_DTYPE.itemsize, dtype=torch.uint8, device="cuda")
    ctx.l1_detect(d_buf.data_ptr() + (P1 - 1) * 32 + 16, T * P1 * 32, P1 * 32, n, T, d_out)
    got = d_out.cpu().numpy().view(A.L1_OUT_DTYPE)
    classes = set()
    for s in range(n):
        xs = x[s].astype(np.float64)
        j = PL.l1_jitter(xs)
        cp = PL.l1_change_point(xs)
        g = got[s]
        assert int(g["n_intervals"]) == len(j), s
        for i, (a, b, basel, wdt) in enumerate(j[:A.L1_MAX_INTERVALS]):
            iv = g["interval"][i]
            assert (int(iv["first"]), int(iv["last"]), int(iv["width"])) == (a, b, wdt), (s, i)
            assert iv["baseline"] == basel
        assert int(g["cp_found"]) == cp[0] and (not cp[0] or int(g["cp_step"]) == cp[1]), s
        assert g["cp_ratio"] == pytest.approx(cp[2], rel=1e-12)
        assert int(g["cls"]) == PL.l1_classify(j, cp)
        classes.add(int(g["cls"]))
    assert {0, 1, 2} <= classes
    # too short for a window / for two segments: stable, nothing found
    d_out.zero_()
    ctx.l1_detect(d_buf.data_ptr() + (P1 - 1) * 32 + 16, T * P1 * 32, P1 * 32, n, 5, d_out)
    g = d_out.cpu().numpy().view(A.L1_OUT_DTYPE)
    assert (g["cls"] == 0).all() and (g["n_intervals"] == 0).all()
    ctx.close()
