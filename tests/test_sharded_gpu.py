"""-m gpu: ONE job sharded by trace rank on ONE device: G shards = G contexts, the
exchange done by the same pack / assemble / diagnose_planes code a multi-GPU run uses (the transport
between the shards is emulated by slicing the send buffers; the world-of-two gloo test covers the
torch.distributed transport).  The merged result must equal the single-job oracle bit for bit."""
import numpy as np
import pytest

from gpu_util import first_diff, run_oracle
from paper_2606_20374_b200.workload import build_workload, scaled

pytestmark = pytest.mark.gpu


def _shard_events(ev, r0, r1):
    """Events of ranks [r0, r1) with the rank field rebased to the shard (input preparation only)."""
    sel = ev[(ev["rank"] >= r0) & (ev["rank"] < r1)].copy()
    sel["rank"] -= r0
    return sel


def _check(merged, ev, dims):
    o, orec, odiag = run_oracle(ev, *dims)
    for k in ("sig_stats", "sig_flags", "span_stats", "span_flags", "rank_score", "step_anomalous"):
        assert (merged[k] == odiag[k]).all(), (k, first_diff(merged[k].view(np.uint8), odiag[k].view(np.uint8)))
    return o, orec


@pytest.mark.parametrize("name,kw,G", [("tiny", {}, 2), ("tiny", {}, 3),
                                        ("mid", dict(n_ranks=37, n_steps=2, n_events=4000), 4),
                                        ("mid", dict(n_ranks=5, n_steps=1, n_events=3000, n_sigs=3), 5)])
@pytest.mark.parametrize("mode", ["a2a", "p2p"])
def test_sharded_job_matches_single_job_oracle(name, kw, G, mode):
    import torch
    from paper_2606_20374_b200 import sharded as Sh
    wl = build_workload(scaled(name, **kw))
    s = wl.spec
    ev = wl.expand_host()
    dims = (s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)
    lay = Sh.Layout(G, s.n_ranks, s.n_steps, s.n_sigs, s.n_phases)
    assert lay.ranks[0][0] == 0 and lay.ranks[-1][1] == s.n_ranks and lay.sigs[-1][1] == s.n_sigs
    shards = [Sh.Shard(lay, g, s.step_base) for g in range(G)]
    recs = []
    for sh in shards:
        se = _shard_events(ev, sh.r0, sh.r1)
        d = torch.from_numpy(se.view(np.uint8).reshape(-1).copy()).cuda() if se.size else None
        sh.aggregate(d, se.size)
        recs.append(sh.ctx.records_to_host(sh.rec))
    if mode == "a2a":
        for sh in shards:
            sh.send.fill_(-1)
            sh.pack_for_all_to_all()
        for d, sh in enumerate(shards):
            # what all_to_all_single delivers to d: source g's d-th split, sources concatenated
            parts = []
            for g, src in enumerate(shards):
                cnt = lay.send_counts(g)
                off = sum(cnt[:d])
                parts.append(src.send[off:off + cnt[d]])
            recv = torch.cat(parts)
            assert recv.numel() == sum(lay.recv_counts(d))
            sig_plane = Sh.assemble_sig_plane(lay, d, recv)
            span_plane = Sh.assemble_span_plane(lay, [x.span_part for x in shards])
            sh.diagnose(sig_plane, span_plane)
    else:
        smax = max(b - a for a, b in lay.sigs)
        sig_planes = [torch.full((lay.T * smax * lay.R,), -1, dtype=torch.int64, device="cuda") for _ in range(G)]
        span_planes = [torch.full((lay.T * (lay.P + 1) * lay.R,), -1, dtype=torch.int64, device="cuda") for _ in range(G)]
        for sh in shards:       # every shard stores its columns into every owner's plane ("peer" pointers)
            sh.pack_into_planes([p.data_ptr() for p in sig_planes], [p.data_ptr() for p in span_planes])
        for d, sh in enumerate(shards):
            sh.diagnose(sig_planes[d], span_planes[d])
    merged = Sh.merge_outputs(lay, [sh.outs_to_host() for sh in shards])
    o, orec = _check(merged, ev, dims)
    # the shards' tables are the single job's table, rank block by rank block (only the header's rank
    # field is shard-relative)
    rb = orec.shape[1]
    for sh, rec in zip(shards, recs):
        want = orec[sh.r0 * s.n_steps: sh.r1 * s.n_steps].copy()
        hdr_rank = want[:, 12:16].view(np.uint32)
        hdr_rank -= sh.r0
        assert (rec == want).all()
    assert sum(sh.ctx.stats()[0] for sh in shards) == o.n_valid
    for sh in shards:
        sh.close()


def test_planes_argument_errors():
    import torch
    from paper_2606_20374_b200 import argus as A
    ctx = A.Argus(4, 2, 6, 2)
    rec = ctx.alloc_records()
    plane = torch.zeros(2 * 6 * 8, dtype=torch.int64, device="cuda")
    span = torch.zeros(2 * 3 * 8, dtype=torch.int64, device="cuda")
    outs = ctx.alloc_diag()

    def code(fn, *a):
        try:
            fn(*a)
        except A.ArgusError as e:
            return e.code
        return A.OK
    ctx.reset(rec)
    assert code(ctx.pack_planes, rec, 0, 6, plane, span, 8, 0) == A.ESTATE      # not finalised
    ctx.phase_times(rec)
    assert code(ctx.pack_planes, rec, 0, 7, plane, span, 8, 0) == A.EINVAL      # sig range
    assert code(ctx.pack_planes, rec, 4, 2, plane, span, 8, 0) == A.EINVAL
    assert code(ctx.pack_planes, rec, 0, 6, plane, span, 8, 5) == A.EINVAL      # columns past the stride
    assert code(ctx.pack_planes, rec, 0, 6, plane.data_ptr() + 4, span, 8, 0) == A.EINVAL
    assert code(ctx.pack_planes, rec, 0, 6, plane, span, 8, 4) == A.OK
    assert code(ctx.diagnose_planes, plane, span, 0, 8, 6, outs) == A.EINVAL    # R = 0
    assert code(ctx.diagnose_planes, plane, span, 9, 8, 6, outs) == A.EINVAL    # stride < R
    assert code(ctx.diagnose_planes, plane, span, 8, 8, 7, outs) == A.EINVAL    # more sigs than the ctx
    assert code(ctx.diagnose_planes, None, span, 8, 8, 6, outs) == A.EINVAL     # sigs without a plane
    big = {k: torch.zeros(v.numel() * 2, dtype=v.dtype, device="cuda") for k, v in outs.items()}
    assert code(ctx.diagnose_planes, plane, span, 8, 8, 6, big) == A.OK
    assert code(ctx.diagnose_planes, None, span, 8, 8, 0, big) == A.OK
    ctx.stats()
    ctx.close()


def test_pack_planes_with_more_steps_than_one_grid_dimension():
    """T > 65535 (the z limit of a grid): the sig-plane export walks the steps inside the kernel."""
    import torch
    from paper_2606_20374_b200 import argus as A
    R, T, S, P = 2, 70000, 3, 1
    steps = np.array([0, 1, 65534, 65535, 65536, 69999], dtype=np.uint32)
    ev = np.zeros(steps.size * R, dtype=A.EVENT_DTYPE)
    ev["rank"] = np.repeat(np.arange(R, dtype=np.uint32), steps.size)
    ev["step"] = np.tile(steps, R)
    ev["sig"] = np.arange(ev.size) % S
    ev["start_ns"] = 1000 + np.arange(ev.size) * 10
    ev["end_ns"] = ev["start_ns"] + 7 + np.arange(ev.size) * 3
    ctx = A.Argus(R, T, S, P)
    rec = ctx.alloc_records()
    ctx.reset(rec)
    ctx.aggregate(torch.from_numpy(ev.view(np.uint8).reshape(-1).copy()).cuda(), ev.size, rec)
    ctx.phase_times(rec)
    sig_plane = torch.full((T * S * R,), -1, dtype=torch.int64, device="cuda")
    span_plane = torch.full((T * (P + 1) * R,), -1, dtype=torch.int64, device="cuda")
    ctx.pack_planes(rec, 0, S, sig_plane, span_plane, R, 0)
    ctx.stats()
    got_sig = sig_plane.cpu().numpy().reshape(T, S, R)
    got_span = span_plane.cpu().numpy().reshape(T, P + 1, R)
    o, _, _ = run_oracle(ev, R, T, S, P, 0)
    cells = o.cells().reshape(R, T, S)
    spans = o.spans().reshape(R, T, P + 1)
    assert (got_sig == cells["sum"].astype(np.int64).transpose(1, 2, 0)).all()
    assert (got_span == spans["span"].astype(np.int64).transpose(1, 2, 0)).all()
    assert int(got_sig[69999].sum()) > 0 and int(got_sig[65536].sum()) > 0
    ctx.close()
