"""-m gpu: argus_diagnose_planes_static, the cross-rank rule for callers that cannot allocate device memory.

Who needs it: a monitor that lives inside the training process it watches.  There the framework's caching
allocator has normally taken the HBM already, so a cudaMalloc made from the side can fail, and one that succeeds
locks the whole device for a moment — in the middle of the iteration being timed.  Such a caller passes buffers it
set aside at start-up and the library brings its own scratch: a 256 KiB array of mark bytes that is part of
libargus.so (ARGUS_STATIC_MAX_SERIES series at most).

What is checked: on the same planes the static entry point writes byte for byte what argus_diagnose_planes (ctx +
workspace) writes — all work is integer, so the tolerance is zero like everywhere else in this suite — for two calls
in a row that share the array.  The first job is full of series that span 2^32 ns or more (those are the ones the
marks exist for); the second has a different geometry and fewer of them, so marks left by the first call would
send the wrong series to the 64-bit pass if the entry point did not clear them.  A sample of series is also
checked against the oracle, and a job beyond the fixed maximum must be refused with ESIZE before anything runs.

This file is named to be collected last: with `pytest -x` a failure here cannot hide the other tests.  It does not
depend on them: the array's address is looked up by the first call in whatever process this runs in."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

KEYS = ("sig_stats", "sig_flags", "span_stats", "span_flags", "rank_score", "step_anomalous")


def _planes(seed, R, stride, T, S, P, wide_every):
    """Seeded [T][S][stride] and [T][P+1][stride] u64 planes; every wide_every-th series gets values 2^33 apart."""
    rng = np.random.default_rng(seed)
    sig = rng.integers(1_000_000, 5_000_000, size=(T, S, stride), dtype=np.uint64)
    span = rng.integers(10_000_000, 11_000_000, size=(T, P + 1, stride), dtype=np.uint64)
    for plane in (sig, span):
        flat = plane.reshape(-1, stride)
        for i in range(0, flat.shape[0], wide_every):
            flat[i, rng.integers(0, R, size=max(1, R // 7))] += np.uint64(1) << np.uint64(33 + i % 20)
    # a few stragglers so that HIGH / LOW flags and the roll-ups are not all zero
    sig[:, :, R // 2] *= np.uint64(3)
    span[:, P, R // 3] *= np.uint64(2)
    return sig, span


def _alloc_outs(torch, R, T, S, P, fill):
    outs = {"sig_stats": torch.empty(T * S * 32, dtype=torch.uint8, device="cuda"),
            "sig_flags": torch.empty(T * S * R, dtype=torch.uint8, device="cuda"),
            "span_stats": torch.empty(T * (P + 1) * 32, dtype=torch.uint8, device="cuda"),
            "span_flags": torch.empty(T * (P + 1) * R, dtype=torch.uint8, device="cuda"),
            "rank_score": torch.empty(T * R, dtype=torch.int32, device="cuda"),
            "step_anomalous": torch.empty(T, dtype=torch.int32, device="cuda")}
    for v in outs.values():
        v.fill_(fill)               # garbage: the call must define every byte
    return outs


def _host(outs):
    return {k: v.cpu().numpy().view(np.uint8).copy() for k, v in outs.items()}


# (R, stride, T, S, P, every n-th series wide): a warp per series, then the block kernel with a padded stride
JOBS = [(37, 37, 3, 29, 4, 2), (300, 304, 2, 11, 2, 5)]


def test_static_entry_matches_ctx_path_on_two_calls_in_a_row():
    import torch
    from oracle import series as oracle_series
    from paper_2606_20374_b200 import argus as A

    for call, (R, stride, T, S, P, wide_every) in enumerate(JOBS):
        sig, span = _planes(100 + call, R, stride, T, S, P, wide_every)
        d_sig = torch.from_numpy(sig.view(np.int64).reshape(-1)).cuda()
        d_span = torch.from_numpy(span.view(np.int64).reshape(-1)).cuda()

        ctx = A.Argus(4, T, S, P)               # the existing path: a ctx whose workspace holds the marks
        want = _alloc_outs(torch, R, T, S, P, 0x5A)
        ctx.diagnose_planes(d_sig, d_span, R, stride, S, want)
        ctx.stats()
        ctx.close()

        got = _alloc_outs(torch, R, T, S, P, 0xA5)
        A.diagnose_planes_static(d_sig, d_span, R, stride, S, T, P, got)
        torch.cuda.synchronize()
        w, g = _host(want), _host(got)
        for k in KEYS:
            assert (g[k] == w[k]).all(), (call, k)

        # and a sample of series against the oracle (wide ones included: index 0 always is)
        stats = g["sig_stats"].view(A.STAT_DTYPE).reshape(T, S)
        flags = g["sig_flags"].reshape(T, S, R)
        for t, s in ((0, 0), (0, 1), (T - 1, S - 1), (T - 1, wide_every % S)):
            med, mad, nh, nl, fl = oracle_series(sig[t, s, :R])
            st = stats[t, s]
            assert (int(st["median"]), int(st["mad"]), int(st["n_high"]), int(st["n_low"])) == (med, mad, nh, nl)
            assert (flags[t, s] == fl).all()
        sstats = g["span_stats"].view(A.STAT_DTYPE).reshape(T, P + 1)
        med, mad, nh, nl, fl = oracle_series(span[0, P, :R])
        assert (int(sstats[0, P]["median"]), int(sstats[0, P]["mad"])) == (med, mad)
        assert int(g["step_anomalous"].view(np.uint32)[0]) == nh


def test_static_entry_refuses_what_the_fixed_array_cannot_hold():
    import torch
    from paper_2606_20374_b200 import argus as A
    R, P = 2, 1
    S = A.STATIC_MAX_SERIES - (P + 1)          # T * (S + P + 1) == the maximum: accepted
    plane = torch.zeros(S * R, dtype=torch.int64, device="cuda")
    span = torch.zeros((P + 1) * R, dtype=torch.int64, device="cuda")
    stats = torch.empty(S * 32, dtype=torch.uint8, device="cuda")
    A.diagnose_planes_static(plane, span, R, R, S, 1, P, {"sig_stats": stats})
    torch.cuda.synchronize()
    assert int(stats.view(torch.int64).abs().sum()) == 0    # medians and MADs of all-zero series
    with pytest.raises(A.ArgusError) as e:                  # one series more: refused, nothing launched
        A.diagnose_planes_static(plane, span, R, R, S, 1, P + 1, {"sig_stats": stats})
    assert e.value.code == A.ESIZE
    with pytest.raises(A.ArgusError) as e:
        A.diagnose_planes_static(plane, span, R, R, S, 2, P, {"sig_stats": stats})
    assert e.value.code == A.ESIZE
    with pytest.raises(A.ArgusError) as e:                  # the argument checks of argus_diagnose_planes
        A.diagnose_planes_static(plane, span, 0, R, S, 1, P, {"sig_stats": stats})
    assert e.value.code == A.EINVAL
    torch.cuda.synchronize()
