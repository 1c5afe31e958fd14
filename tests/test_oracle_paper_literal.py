"""CPU-only pins of oracle/paper_literal.py (the paper-literal float algorithms, SURVEY §8(f) NEXT-1..3)
against what the paper and the mathematics fix: closed forms, invariants, special cases that reduce to a
textbook or library routine, brute force on tiny inputs.  Each pin is chosen so that a plausible mistake
(a dropped 1/h, a wrong sign, n instead of n - 1, a transposed argument) fails it."""
import math
import random

import numpy as np
import pytest

from oracle import paper_literal as PL


# ---- NEXT-1: the fine grid --------------------------------------------------------------------------
def test_fine_bin_is_floor_8_log2_exactly():
    # thresholds: the smallest d of bin k is ceil(2^(k/8)); checked with Python big ints on both sides of
    # every threshold, no floating point involved
    for k in range(1, 256):
        # integer 8th root: largest d with d^8 < 2^k
        lo, hi = 1, 1 << 33
        while lo < hi:
            mid = (lo + hi + 1) // 2
            if mid ** 8 < (1 << k):
                lo = mid
            else:
                hi = mid - 1
        # lo is the last integer below the threshold 2^(k/8), lo + 1 the first at or above it (the lowest
        # bins hold no integer at all: 2 is already bin 8)
        assert PL.fine_bin(lo) < k <= PL.fine_bin(lo + 1), k
        assert PL.fine_bin(lo + 1) == min(255, ((lo + 1) ** 8).bit_length() - 1)
    assert PL.fine_bin(0) == 0 and PL.fine_bin(1) == 0 and PL.fine_bin(2) == 8 and PL.fine_bin(3) == 12
    assert PL.fine_bin(2**32 - 1) == 255 and PL.fine_bin(2**40) == 255
    # the coarse 32-bucket grid is the fine one summed 8 at a time (R4 vs R23)
    rnd = random.Random(1)
    for _ in range(2000):
        d = rnd.getrandbits(rnd.randint(1, 32))
        assert PL.fine_bin(d) // 8 == max(d.bit_length() - 1, 0)


def _hist_from_log_samples(xs):
    """Samples given as log2-durations -> the 256-bin histogram of the rounded durations."""
    h = np.zeros(256, dtype=np.int64)
    for v in xs:
        h[PL.fine_bin(int(round(2.0 ** v)))] += 1
    return h


def test_scott_bandwidth_closed_form():
    # two bins, a and b, with counts m each: mean = midpoint, sample variance = (n/(n-1)) * (delta/2)^2
    h = np.zeros(256, dtype=np.int64)
    h[100], h[116] = 500, 500
    f, bw, bounds, cl = PL.kde_clusters(h)
    delta = 16 / 8 * math.log(2.0)
    sigma = math.sqrt(1000 / 999.0) * delta / 2
    assert bw == pytest.approx(1.06 * sigma * 1000 ** -0.2, rel=1e-12)
    # density integrates to one over the grid (the 1/h factor of eq. 1, R22): Riemann sum with the grid step
    assert f.sum() * (math.log(2.0) / 8) == pytest.approx(1.0, rel=1e-3)
    # ... and is symmetric about the midpoint bin 108
    assert np.allclose(f[100:117], f[100:117][::-1], rtol=1e-12)


def test_two_separated_modes_one_valley_and_analytic_percentiles():
    rnd = np.random.default_rng(7)
    a = rnd.normal(14.0, 0.05, 6000)          # log2 ns: ~16 us
    b = rnd.normal(18.0, 0.05, 4000)          # 16x slower ("differ by several multiples")
    h = _hist_from_log_samples(np.concatenate([a, b]))
    f, bw, bounds, cl = PL.kde_clusters(h)
    assert len(bounds) == 1 and 14 * 8 < bounds[0] < 18 * 8
    assert [c[0] for c in cl] == [6000, 4000] and sum(c[0] for c in cl) == h.sum()
    # p50 of N(14, 0.05) in log2 is 14.0 -> bin 112 (within one bin of rounding); p99 = 14 + 2.326 * 0.05
    assert abs(cl[0][1] - 112) <= 1 and abs(cl[0][2] - int((14 + 2.326 * 0.05) * 8)) <= 1
    assert abs(cl[1][1] - 144) <= 1 and abs(cl[1][2] - int((18 + 2.326 * 0.05) * 8)) <= 1
    assert PL.bin_value_ns(112) == pytest.approx(2 ** 14.0625)


def test_unimodal_and_degenerate_inputs_give_one_cluster():
    rnd = np.random.default_rng(3)
    h = _hist_from_log_samples(rnd.normal(15.5, 0.15, 5000))
    f, bw, bounds, cl = PL.kde_clusters(h)
    assert bounds == [] and len(cl) == 1 and cl[0][0] == 5000
    # brute-force percentiles of the binned data
    bins = np.repeat(np.arange(256), h)
    assert cl[0][1] == bins[math.ceil(0.5 * 5000) - 1] and cl[0][2] == bins[math.ceil(0.99 * 5000) - 1]
    # one sample, all samples in one bin, empty
    for hh, want in ((np.eye(1, 256, 77, dtype=np.int64)[0], [(1, 77, 77)]),
                     (np.eye(1, 256, 9, dtype=np.int64)[0] * 50, [(50, 9, 9)]),
                     (np.zeros(256, dtype=np.int64), [])):
        f, bw, bounds, cl = PL.kde_clusters(hh)
        assert bw == 0.0 and bounds == [] and cl == want


def test_filters_reject_noise_valleys():
    # a tiny satellite (3 samples) far from a big mode: the valley exists but the cluster-level filter (R28)
    # rejects it
    h = np.zeros(256, dtype=np.int64)
    h[100:104] = [400, 900, 800, 300]
    h[160] = 3
    f, bw, bounds, cl = PL.kde_clusters(h)
    assert bounds == [] and cl[0][0] == 2403
    # the spacing filter (R29) acts between adjacent RETAINED boundaries: three spikes two bins apart give the
    # candidates 101 and 103, a quarter octave apart (< half an octave): the second is dropped
    h2 = np.zeros(256, dtype=np.int64)
    h2[100], h2[102], h2[104] = 1000, 1000, 1000
    f, bw, bounds, cl = PL.kde_clusters(h2)
    assert bounds == [101] and [c[0] for c in cl] == [1000, 2000]
    assert PL.kde_clusters(h2, min_gap_bins=0)[2] == [101, 103]
    # three well separated modes: two boundaries, counts add up, boundaries ascending
    h3 = np.zeros(256, dtype=np.int64)
    h3[80:83] = [300, 500, 300]
    h3[120:123] = [200, 400, 200]
    h3[170:173] = [100, 300, 100]
    f, bw, bounds, cl = PL.kde_clusters(h3)
    assert len(bounds) == 2 and bounds[0] < bounds[1] and [c[0] for c in cl] == [1100, 800, 500]


def test_fine_histograms_bruteforce_and_coarse_consistency():
    from helpers import make_events
    from oracle import Oracle
    rnd = random.Random(5)
    rows = []
    for _ in range(3000):
        a = rnd.randrange(10**6)
        d = int(rnd.lognormvariate(9, 2)) if rnd.random() < 0.97 else -5
        rows.append((rnd.randrange(3), 7 + rnd.randrange(2), rnd.randrange(5 + (rnd.random() < 0.02)), 0, rnd.randrange(2), a, a + d))
    ev = make_events(rows)
    fh = PL.fine_histograms(ev, 3, 2, 5, 2, 7)
    o = Oracle(3, 2, 5, 2, 7)
    o.aggregate(ev)
    cells = o.cells()
    assert fh.sum() == o.n_valid
    assert (fh.reshape(3, 2, 5, 32, 8).sum(axis=4) == cells["hist"]).all()     # 8 fine bins per log2 bucket


# ---- NEXT-2 -------------------------------------------------------------------------------------------
def test_lognormal_cdf_hits_its_defining_percentiles():
    xs = np.array([50_000.0, 80_000.0])
    F = PL.mixture_cdf([(10, 50_000.0, 80_000.0)], xs)
    assert F[0] == pytest.approx(0.5, abs=1e-15)                   # mu = ln p50
    assert F[1] == pytest.approx(0.99, abs=2e-5)                   # z_0.99 = 2.326 (Phi(2.326) = 0.98999)
    assert PL.normal_cdf(np.array([0.0, 1.0]))[1] == pytest.approx(0.8413447460685429, rel=1e-14)
    # mixture weights: 3:1
    F2 = PL.mixture_cdf([(3, 10.0, 10.0), (1, 1000.0, 1000.0)], np.array([5.0, 20.0, 2000.0]))
    assert list(F2) == [0.0, 0.75, 1.0]
    assert list(PL.mixture_cdf([], xs)) == [0.0, 0.0]


def test_w1_of_shifted_steps_is_the_shift_and_metric_properties():
    xs = PL.log_grid(1.0, 1e6, 20001)
    assert xs[0] == pytest.approx(1.0) and xs[-1] == pytest.approx(1e6) and np.allclose(xs[1:] / xs[:-1], xs[1] / xs[0])
    Fa = PL.mixture_cdf([(5, 1000.0, 1000.0)], xs)                 # step at 1000
    Fb = PL.mixture_cdf([(7, 3000.0, 3000.0)], xs)                 # step at 3000
    assert PL.w1(Fa, Fb, xs) == pytest.approx(2000.0, rel=2e-3)    # area between two unit steps
    assert PL.w1(Fa, Fa, xs) == 0.0 and PL.w1(Fa, Fb, xs) == PL.w1(Fb, Fa, xs)
    Fc = PL.mixture_cdf([(1, 2000.0, 2600.0)], xs)
    assert PL.w1(Fa, Fb, xs) <= PL.w1(Fa, Fc, xs) + PL.w1(Fc, Fb, xs) + 1e-9
    # W1 between two log-normals with the same sigma = difference of their means e^(mu + sigma^2/2) (they are
    # stochastically ordered, so W1 = |E a - E b|)
    sg = (math.log(1500.0) - math.log(1000.0)) / 2.326
    Fd = PL.mixture_cdf([(1, 1000.0, 1500.0)], xs)
    Fe = PL.mixture_cdf([(1, 1200.0, 1800.0)], xs)
    assert PL.w1(Fd, Fe, xs) == pytest.approx(200.0 * math.exp(sg * sg / 2), rel=2e-3)


def test_l3_scores_flag_the_shifted_rank():
    rnd = random.Random(2)
    R = 24
    tr = [[(100, 50_000.0 * (1 + 0.01 * rnd.random()), 70_000.0 * (1 + 0.01 * rnd.random())),
           (40, 400_000.0, 500_000.0)] for _ in range(R)]
    tr[5] = [(100, 75_000.0, 105_000.0), (40, 400_000.0, 500_000.0)]     # 1.5x slower first mode
    xs, F, W, score, q1, q3, fence, flags = PL.l3_scores(tr, n_grid=128, alpha=1.5)
    assert W.shape == (R, R) and np.allclose(W, W.T) and (np.diag(W) == 0).all()
    # mean W1 to the others, by the plain double loop
    for r in range(R):
        assert score[r] == pytest.approx(sum(W[r, b] for b in range(R) if b != r) / (R - 1), rel=1e-12)
    s = sorted(score)
    assert q1 == pytest.approx(s[5] + 0.75 * (s[6] - s[5]), rel=1e-12)     # numpy linear interpolation, n = 24
    assert fence == pytest.approx(q3 + 1.5 * (q3 - q1))
    # recall, not precision (a tight IQR also flags the largest natural deviations): the shifted rank is
    # flagged, its score dwarfs everybody else's, and a generous alpha leaves it alone above the fence
    assert flags[5] == 1 and score[5] > 10 * np.median(score) and int(np.argmax(score)) == 5
    assert list(np.nonzero(PL.l3_scores(tr, n_grid=128, alpha=20.0)[7])[0]) == [5]
    assert xs[0] == pytest.approx(0.5 * min(t[0][1] for t in tr)) and xs[-1] == pytest.approx(1_000_000.0)


# ---- NEXT-3 -------------------------------------------------------------------------------------------
def test_l2_cv_and_z_closed_forms():
    # group 0: 1, 2, 3, 4, 5 -> mu 3, sigma sqrt(2.5) (n - 1), CV 0.527: severe; z of 5 = 2/sqrt(2.5)
    x = np.array([1, 2, 3, 4, 5, 100, 100, 100, 102, 7], dtype=np.float64)
    g = np.array([0, 0, 0, 0, 0, 1, 1, 1, 1, 2])
    out, z, flag = PL.l2_groups(x, g, z_thr=1.2)
    n, mu, sigma, cv, cls = out[0]
    assert (n, mu) == (5, 3.0) and sigma == pytest.approx(math.sqrt(2.5)) and cls == 2
    assert z[4] == pytest.approx(2 / math.sqrt(2.5)) and z[0] == pytest.approx(-2 / math.sqrt(2.5))
    n, mu, sigma, cv, cls = out[1]
    assert mu == 100.5 and sigma == pytest.approx(1.0) and cv == pytest.approx(1 / 100.5) and cls == 0
    assert out[2] == (1, 7.0, 0.0, 0.0, 0) and z[9] == 0.0               # a group of one (R34)
    assert list(flag) == [0, 0, 0, 0, 1, 0, 0, 0, 1, 0]
    # class edges: CV = 0.02 is mild, 0.05 is severe
    for cv_t, cls_t in ((0.0199, 0), (0.0201, 1), (0.0499, 1), (0.0501, 2)):
        s = cv_t * 100 * math.sqrt(0.5)          # two points mu +- s/sqrt(2)... sample sigma of {100-a, 100+a} = a*sqrt(2)
        out, _, _ = PL.l2_groups(np.array([100 - s, 100 + s]), np.array([0, 0]))
        assert out[0][4] == cls_t and out[0][3] == pytest.approx(cv_t, rel=1e-9)


def test_l1_jitter_recovers_a_narrow_spike():
    # a spike much narrower than W smears the candidate region to >= W; phase 2 recovers its
    # true width
    x = [100.0] * 64
    x[30], x[31], x[32] = 190.0, 200.0, 180.0
    got = PL.l1_jitter(x, W=8, theta=1.5, beta=1.25)
    assert got == [(23, 39, 100.0, 3)]
    assert PL.l1_jitter([100.0] * 64) == [] and PL.l1_jitter([100.0] * 5, W=8) == []
    # two spikes far apart: two intervals; close together: merged
    y = [100.0] * 64
    y[10] = y[50] = 300.0
    assert [(a, b, w) for a, b, _, w in PL.l1_jitter(y)] == [(3, 17, 1), (43, 57, 1)]
    y[20] = 300.0
    assert [(a, b) for a, b, _, _ in PL.l1_jitter(y)][0] == (3, 27)
    # the gate is a RATIO: scaling the series changes nothing but the baseline
    assert [(a, b, w) for a, b, _, w in PL.l1_jitter([7 * v for v in x])] == [(23, 39, 3)]
    assert PL.median_f64([3, 1, 2]) == 2.0 and PL.median_f64([4, 1, 3, 2]) == 2.5


def test_l1_change_point_finds_the_step():
    x = [100.0 + (i % 3) for i in range(40)] + [130.0 + (i % 3) for i in range(24)]
    found, t, ratio = PL.l1_change_point(x)
    assert (found, t) == (1, 40) and ratio == pytest.approx(131.0 / 101.0, rel=1e-3)
    assert PL.l1_change_point([100.0] * 64)[0] == 0                       # no regression
    assert PL.l1_change_point([100.0] * 40 + [105.0] * 24)[0] == 0        # below the minimum ratio 1.1
    noisy = [100.0 if i % 2 else 140.0 for i in range(40)] + [260.0] * 24
    assert PL.l1_change_point(noisy)[0] == 0                              # left side not stable (sigma/mu >= 0.05)
    assert PL.l1_change_point(x[:6])[0] == 0                              # too short for two segments of 4
    assert PL.l1_classify(PL.l1_jitter(x), PL.l1_change_point(x)) in (2, 3)
    assert PL.l1_classify([], (0, 0, 0.0)) == 0


def test_plateau_valley_belongs_to_its_left_edge():
    """R27 ("local minima ... as candidate cluster boundaries"): bin j is a valley when f[j] < f[j-1] and
    f[j] <= f[j+1], so a flat valley floor yields ONE boundary, at its left edge.  Two equal modes an odd number of
    bins apart put the floor on two bins with exactly equal density (checked, not assumed): a rule strict on both
    sides would find no valley at all, a rule lax on the left would pick the right-hand bin."""
    for per_octave, n_bins, b1, b2 in ((1, 32, 10, 15), (8, 256, 40, 53)):
        h = np.zeros(n_bins, dtype=np.int64)
        h[b1] = h[b2] = 100
        f, _, bounds, clusters = PL.kde_clusters(h, per_octave=per_octave, min_gap_bins=0)
        j = (b1 + b2) // 2
        assert f[j] == f[j + 1] and f[j] < f[j - 1] and f[j + 1] < f[j + 2]      # a two-bin plateau at the bottom
        assert bounds == [j]
        assert clusters == [(100, b1, b1), (100, b2, b2)]


def test_l1_classify_exact_values():
    """PAPER.md:222 "stable, jitter, regression, or both": bit 0 = some jitter interval of non-zero effective width,
    bit 1 = a change point was found."""
    spike = [(10, 17, 100.0, 3)]           # (first, last, baseline, width)
    none_wide = [(10, 17, 100.0, 0)]       # a candidate whose run above beta x baseline is empty: not jitter
    assert PL.l1_classify([], (0, 0, 0.0)) == 0
    assert PL.l1_classify(none_wide, (0, 0, 0.0)) == 0
    assert PL.l1_classify(spike, (0, 0, 0.0)) == 1
    assert PL.l1_classify([], (1, 40, 1.3)) == 2
    assert PL.l1_classify(none_wide, (1, 40, 1.3)) == 2
    assert PL.l1_classify(spike + none_wide, (1, 40, 1.3)) == 3
    # and on real series: a clean step is a regression only, a spike on a flat line jitter only, both together both
    step = [100.0 + (i % 3) for i in range(40)] + [130.0 + (i % 3) for i in range(24)]
    assert PL.l1_classify(PL.l1_jitter(step), PL.l1_change_point(step)) == 2
    flat = [100.0] * 64
    spiky = list(flat)
    spiky[30] = spiky[31] = 200.0
    assert PL.l1_classify(PL.l1_jitter(spiky), PL.l1_change_point(spiky)) == 1
    assert PL.l1_classify(PL.l1_jitter(flat), PL.l1_change_point(flat)) == 0
