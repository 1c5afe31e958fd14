"""CPU ORACLE of the paper-literal float algorithms —
TEST INFRASTRUCTURE, NOT PRODUCT.  numpy / plain Python in fp64, step by step in the paper's order and
notation; no blocking, fusion or reordering beyond what the passages state.  Where the paper leaves a
constant or a rule open, the reading of DESIGN.md §3 (R23-R34) is taken and named at the spot.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this; it shares no code
with paper_2606_20374_b200 and imports nothing from it.

PAPER.md = /root/reference/PAPER.md (arxiv/paper_2606_20374).

Pins (tests/test_oracle_paper_literal.py, -m "not gpu"): Scott bandwidth closed form; two well separated
modes -> exactly one valley and the analytic bin of p50 / p99; a unimodal sample -> one cluster; counts
sum to n; fine_bin against Python big-int bit lengths of d^8; the log-normal CDF against the error
function at the median / p99 (F = 0.5, 0.99); W1 of two shifted step CDFs = the shift; W1 symmetry,
identity and the triangle inequality; the mean-W1 score against the O(R^2) double loop; numpy's
percentile for Q1 / Q3; CV / z closed forms on hand-made groups; jitter and change-point on hand-made
series with known answers.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

import numpy as np

# ================================================================================================
# NEXT-1  online statistical compression: log transform -> KDE on an equally spaced grid -> valleys ->
#         two filters -> per-cluster (count, p50, p99)                      PAPER.md:176-198 (§5.2, eq. 1)
# ================================================================================================
FINE_PER_OCTAVE = 8          # R23: the "equally-spaced grid" in log-duration: 8 bins per octave, 256 bins
FINE_BINS = 256              #      over [1, 2^32) ns (0 and 1 ns share bin 0; >= 2^32 ns clamps to 255)
SCOTT = 1.06                 # PAPER.md:182 "h = 1.06 * sigma * n^(-1/5)"


def fine_bin(d: int) -> int:
    """R23: bin(d) = floor(8 * log2(d)) clamped to [0, 255], as an EXACT integer rule:
    the largest k with 2^k <= d^8 (Python big ints; no floating point decides a bin)."""
    if d <= 1:
        return 0
    return min(FINE_BINS - 1, (d ** 8).bit_length() - 1)


def fine_histograms(events: np.ndarray, R: int, T: int, S: int, P: int, step_base: int) -> np.ndarray:
    """[R][T][S][256] counts of the valid events (validity R2, R3 as in the integer path)."""
    h = np.zeros((R, T, S, FINE_BINS), dtype=np.uint32)
    for e in events:
        r, st, s, ph = int(e["rank"]), int(e["step"]), int(e["sig"]), int(e["phase"])
        a, b = int(e["start_ns"]), int(e["end_ns"])
        t = st - step_base
        if a < 0 or b < a or r >= R or t < 0 or t >= T or s >= S or ph >= P:
            continue
        h[r, t, s, fine_bin(b - a)] += 1
    return h


def grid_points(n_bins: int, per_octave: int) -> np.ndarray:
    """Log-duration (natural log of ns) at the centre of every bin of the equally spaced grid."""
    return (np.arange(n_bins, dtype=np.float64) + 0.5) / per_octave * math.log(2.0)


def kde_clusters(hist: Sequence[int], per_octave: int = FINE_PER_OCTAVE, min_count: int = 8,
                 min_frac: float = 0.02, min_gap_bins: int = FINE_PER_OCTAVE // 2, max_clusters: int = 8):
    """One (kernel, rank, window) histogram on the equally spaced log grid -> clusters.
    Returns (density f[n_bins], h, boundaries (bin indices), clusters [(count, p50_bin, p99_bin)]).

    PAPER.md:178 "applies a logarithmic transformation to the raw durations, then computes the KDE density
    function on an equally-spaced grid": the samples are the bin centres x_b weighted by the counts (R24:
    binned KDE), the grid is the same bin centres.
    eq. (1) with the 1/h factor restored (R22): f(x) = 1/(n h) * sum_b c_b K((x - x_b)/h), K = N(0, 1) pdf.
    PAPER.md:182 Scott's rule h = 1.06 sigma n^(-1/5); sigma = sample standard deviation (n - 1) of the
    weighted samples (R25); n < 2 or every sample in ONE grid bin (sigma = 0) -> no density, one cluster
    (R26; tested on the occupied range, an integer comparison, not on a rounded sigma).
    PAPER.md:182 "All local minima on the density curve are identified as candidate cluster boundaries":
    bin j strictly inside the occupied range with f[j] < f[j-1] and f[j] <= f[j+1] (R27).
    "cluster-level filtering requires that both sides of each valley contain sufficient samples" (R28): left
    to right, a candidate is kept when the samples since the previous kept boundary and the samples to its
    right both number >= max(min_count, min_frac * n); the boundary belongs to the right-hand cluster.
    "spacing filtering requires that the duration difference between adjacent retained boundaries is
    sufficiently significant" (R29): a kept boundary must lie >= min_gap_bins grid steps (half an octave, a
    factor 1.41 in duration) after the previous kept one — counted in grid steps so that the decision is an
    integer comparison.
    At most max_clusters clusters (a fixed-size output slot): once max_clusters - 1 boundaries are kept, the
    last cluster takes the rest.
    PAPER.md:182-194 per cluster: count, p50, p99 — the bins where the cluster's cumulative count first
    reaches ceil(0.5 count) and ceil(0.99 count) (R30: bin-quantised percentiles)."""
    c = np.asarray(hist, dtype=np.float64)
    nb = c.size
    n = float(c.sum())
    x = grid_points(nb, per_octave)
    f = np.zeros(nb, dtype=np.float64)
    if n == 0:
        return f, 0.0, [], []
    occ = np.nonzero(c)[0]
    lo, hi = int(occ[0]), int(occ[-1])
    h = 0.0
    bounds: List[int] = []
    if n >= 2:
        mean = float((c * x).sum() / n)
        var = float((c * (x - mean) ** 2).sum() / (n - 1.0))
        sigma = math.sqrt(var)
        if hi > lo:
            h = SCOTT * sigma * n ** (-0.2)
            for j in range(nb):
                u = (x[j] - x) / h
                f[j] = float((c * np.exp(-0.5 * u * u)).sum()) / (n * h * math.sqrt(2.0 * math.pi))
            need = max(float(min_count), min_frac * n)
            prev = lo                   # first bin of the current cluster
            for j in range(lo + 1, hi):
                if f[j] < f[j - 1] and f[j] <= f[j + 1]:
                    left = float(c[prev:j].sum())
                    right = float(c[j:hi + 1].sum())
                    if left >= need and right >= need and (not bounds or j - bounds[-1] >= min_gap_bins) \
                            and len(bounds) + 1 < max_clusters:
                        bounds.append(j)
                        prev = j
    clusters = []
    edges = [lo] + bounds + [hi + 1]
    for a, b in zip(edges[:-1], edges[1:]):
        seg = c[a:b]
        cnt = int(seg.sum())
        if cnt == 0:
            continue
        cum = np.cumsum(seg)
        p50 = a + int(np.searchsorted(cum, math.ceil(0.5 * cnt), side="left"))
        p99 = a + int(np.searchsorted(cum, math.ceil(0.99 * cnt), side="left"))
        clusters.append((cnt, p50, p99))
    return f, h, bounds, clusters


def bin_value_ns(b: int, per_octave: int = FINE_PER_OCTAVE) -> float:
    """Duration (ns) a bin stands for: its geometric centre 2^((b + 0.5) / per_octave)."""
    return 2.0 ** ((b + 0.5) / per_octave)


# ================================================================================================
# NEXT-2  L3: log-normal mixture CDF (eq. 2) -> pairwise W1 on a log-uniform grid (eq. 3) -> mean-W1
#         deviation score -> IQR upper fence (eq. 4)                           PAPER.md:234-251 (§6.2)
# ================================================================================================
Z99 = 2.326                  # PAPER.md:234 "z_0.99 = 2.326"


def normal_cdf(z: np.ndarray) -> np.ndarray:
    return 0.5 * np.array([math.erfc(-float(v) / math.sqrt(2.0)) for v in np.ravel(z)]).reshape(np.shape(z))


def mixture_cdf(triples: Sequence[Tuple[float, float, float]], xs: np.ndarray) -> np.ndarray:
    """eq. (2): F(x) = sum_c count_c / sum count * Phi((ln x - mu_c) / sigma_c), mu_c = ln p50_c,
    sigma_c = (ln p99_c - ln p50_c) / 2.326.  sigma_c = 0 (p99 = p50) -> a step at p50 (R31).
    No clusters (the rank never ran the kernel) -> F = 0 everywhere (R31)."""
    F = np.zeros(xs.shape, dtype=np.float64)
    tot = float(sum(t[0] for t in triples))
    if tot == 0:
        return F
    lx = np.log(xs)
    for cnt, p50, p99 in triples:
        if cnt == 0:
            continue
        mu = math.log(p50)
        sg = (math.log(p99) - mu) / Z99
        if sg > 0.0:
            F += cnt / tot * normal_cdf((lx - mu) / sg)
        else:
            F += cnt / tot * (lx >= mu)
    return F


def log_grid(x_lo: float, x_hi: float, n: int) -> np.ndarray:
    """"log-uniform grid": n points, equal ratios, from x_lo to x_hi."""
    return np.exp(np.log(x_lo) + (np.log(x_hi) - np.log(x_lo)) * np.arange(n, dtype=np.float64) / (n - 1))


def w1(Fa: np.ndarray, Fb: np.ndarray, xs: np.ndarray) -> float:
    """eq. (3) by "trapezoidal numerical integration on a log-uniform grid"."""
    d = np.abs(Fa - Fb)
    return float((0.5 * (d[1:] + d[:-1]) * (xs[1:] - xs[:-1])).sum())


def l3_scores(rank_triples: Sequence[Sequence[Tuple[float, float, float]]], n_grid: int = 256, alpha: float = 1.5):
    """One (kernel) key over R ranks: rank_triples[r] = that rank's clusters.
    Grid (R32): log-uniform, n_grid points from 0.5 * the smallest p50 to 2 * the largest p99 over all ranks.
    Returns (xs, F [R][n_grid], W [R][R], score [R] = mean W1 to the other ranks, q1, q3,
    fence = Q3 + alpha (Q3 - Q1) (eq. 4; R33: alpha = 1.5, quartiles by linear interpolation), flags [R])."""
    R = len(rank_triples)
    p50s = [t[1] for tr in rank_triples for t in tr if t[0] > 0]
    p99s = [t[2] for tr in rank_triples for t in tr if t[0] > 0]
    if not p50s:
        z = np.zeros(R)
        return np.ones(n_grid), np.zeros((R, n_grid)), np.zeros((R, R)), z, 0.0, 0.0, 0.0, np.zeros(R, dtype=np.uint8)
    xs = log_grid(0.5 * min(p50s), 2.0 * max(p99s), n_grid)
    F = np.stack([mixture_cdf(tr, xs) for tr in rank_triples])
    W = np.zeros((R, R), dtype=np.float64)
    for a in range(R):
        for b in range(R):
            W[a, b] = w1(F[a], F[b], xs)
    score = W.sum(axis=1) / max(1, R - 1)
    q1, q3 = np.percentile(score, [25.0, 75.0])
    fence = q3 + alpha * (q3 - q1)
    return xs, F, W, score, float(q1), float(q3), float(fence), (score > fence).astype(np.uint8)


# ================================================================================================
# NEXT-3  L2: CV + z-score within a parallelism group (eq. 5, Table 3)
#         L1: sliding-window ratio-gated jitter detection, full-scan change point
# ================================================================================================
def l2_groups(xbar: np.ndarray, group: np.ndarray, z_thr: float = 3.0):
    """xbar[r] = average duration of one event on rank r in the window; group[r] = id of r's group in the
    parallelism dimension the event is routed to (Table 3).  eq. (5): mu_G, sigma_G (|G| - 1), CV = sigma/mu,
    classes balanced < 0.02 <= mild < 0.05 <= severe, z_r = (x_r - mu_G)/sigma_G, straggler
    when z_r > z_thr (R34: threshold 3).  |G| = 1, sigma = 0 or mu = 0 -> CV = 0, z = 0 (R34).
    Returns (per-group dict id -> (n, mu, sigma, cv, cls), z[R], flag[R])."""
    xbar = np.asarray(xbar, dtype=np.float64)
    z = np.zeros(xbar.size, dtype=np.float64)
    out = {}
    for g in sorted(set(int(v) for v in group)):
        idx = np.nonzero(group == g)[0]
        n = idx.size
        mu = float(xbar[idx].sum() / n)
        sigma = math.sqrt(float(((xbar[idx] - mu) ** 2).sum() / (n - 1))) if n > 1 else 0.0
        cv = sigma / mu if (mu > 0.0 and sigma > 0.0) else 0.0
        cls = 0 if cv < 0.02 else (1 if cv < 0.05 else 2)
        if sigma > 0.0:
            z[idx] = (xbar[idx] - mu) / sigma
        out[g] = (n, mu, sigma, cv, cls)
    return out, z, (z > z_thr).astype(np.uint8)


def median_f64(v: Sequence[float]) -> float:
    s = sorted(float(a) for a in v)
    n = len(s)
    return 0.0 if n == 0 else (s[n // 2] if n % 2 else 0.5 * (s[n // 2 - 1] + s[n // 2]))


def l1_jitter(x: Sequence[float], W: int = 8, theta: float = 1.5, beta: float = 1.25):
    """PAPER.md:472.  Phase 1: a window of width W slides point by point; r = max/min of the window; windows
    with r > theta are candidates; adjacent or overlapping candidates merge into intervals [a, b] (inclusive
    point indices).  Phase 2: baseline = median of the points outside the interval; effective width = the
    longest run of points inside it with x > beta * baseline (R35: W = 8, theta = 1.5, "significantly
    exceed" = 1.25 x).  Returns [(a, b, baseline, width)]."""
    x = [float(v) for v in x]
    T = len(x)
    cand = []
    for i in range(0, T - W + 1):
        w = x[i:i + W]
        if max(w) > theta * min(w):
            cand.append((i, i + W - 1))
    merged: List[List[int]] = []
    for a, b in cand:
        if merged and a <= merged[-1][1] + 1:
            merged[-1][1] = max(merged[-1][1], b)
        else:
            merged.append([a, b])
    out = []
    for a, b in merged:
        base = median_f64(x[:a] + x[b + 1:])
        best = run = 0
        for t in range(a, b + 1):
            run = run + 1 if x[t] > beta * base else 0
            best = max(best, run)
        out.append((a, b, base, best))
    return out


def l1_change_point(x: Sequence[float], min_seg: int = 4, ratio_min: float = 1.1, rsd_max: float = 0.05):
    """PAPER.md:474-476.  Every split t (left = x[:t], right = x[t:], both >= min_seg points): mu_L, mu_R,
    sigma/mu of both sides (sample standard deviation, as eq. 5); valid when mu_R / mu_L > ratio_min and both
    relative deviations < rsd_max (R36: 4 points, 1.1, 0.05); the valid split with the largest ratio wins
    (the earliest among equals).  Returns (found, t, ratio)."""
    x = np.asarray(x, dtype=np.float64)
    T = x.size
    best = (0, 0, 0.0)
    for t in range(min_seg, T - min_seg + 1):
        L, Rr = x[:t], x[t:]
        muL, muR = float(L.sum() / L.size), float(Rr.sum() / Rr.size)
        if muL <= 0.0 or muR <= 0.0:
            continue
        sL = math.sqrt(float(((L - muL) ** 2).sum() / (L.size - 1)))
        sR = math.sqrt(float(((Rr - muR) ** 2).sum() / (Rr.size - 1)))
        ratio = muR / muL
        if ratio > ratio_min and sL / muL < rsd_max and sR / muR < rsd_max and ratio > best[2]:
            best = (1, t, ratio)
    return best


def l1_classify(jitter, cp) -> int:
    """stable (0), jitter (1), regression (2), or both (3)."""
    return (1 if any(w > 0 for _, _, _, w in jitter) else 0) | (2 if cp[0] else 0)
