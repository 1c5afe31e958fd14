"""-m gpu: tables a ctx did not aggregate (include/argus.h, "Ownership of a table").  argus_diagnose takes the sig
series of the ctx's OWN table from the sum plane of its workspace and those of any other table from the record
bytes; these tests run that second gather (never reached by the other parity tests) against the oracle, for both
selection geometries (a warp per series, a CTA per series), and the argus_forget protocol for a buffer that is
re-used under a ctx's feet."""
import numpy as np
import pytest

from gpu_util import first_diff, run_oracle
from paper_2606_20374_b200.workload import build_workload, scaled

pytestmark = pytest.mark.gpu

KEYS = ("sig_stats", "sig_flags", "span_stats", "span_flags", "rank_score", "step_anomalous")


def _events(name, **kw):
    wl = build_workload(scaled(name, **kw))
    s = wl.spec
    return wl.expand_host(), (s.n_ranks, s.n_steps, s.n_sigs, s.n_phases, s.step_base)


def _aggregate(ctx, ev, rec):
    import torch
    d = torch.from_numpy(ev.view(np.uint8).reshape(-1).copy()).cuda()
    ctx.reset(rec)
    ctx.aggregate(d, ev.size, rec)
    ctx.phase_times(rec)
    ctx.stats()


def _diag(ctx, rec):
    import torch
    outs = ctx.alloc_diag()
    for v in outs.values():
        v.fill_(0x5A if v.dtype == torch.uint8 else 0x5A5A5A5A)
    ctx.diagnose(rec, outs)
    ctx.stats()
    return ctx.diag_to_host(outs)


def _same(got, want):
    for k in KEYS:
        assert (got[k] == want[k]).all(), (k, first_diff(got[k].view(np.uint8), want[k].view(np.uint8)))


@pytest.mark.parametrize("name,kw", [("tiny", {}), ("mid", dict(n_ranks=300, n_steps=2, n_events=1500, n_sigs=40))])
def test_diagnose_of_a_table_another_ctx_aggregated(name, kw):
    from paper_2606_20374_b200 import argus as A
    ev, dims = _events(name, **kw)
    a = A.Argus(*dims)
    rec = a.alloc_records()
    _aggregate(a, ev, rec)
    _, _, odiag = run_oracle(ev, *dims)
    _same(_diag(a, rec), odiag)                  # own table: sum plane
    b = A.Argus(*dims)                           # never reset: every table is foreign to it
    _same(_diag(b, rec), odiag)                  # record gather
    # the record-only consumers accept the foreign table too
    import torch
    out = torch.empty(b.sparse_bound(), dtype=torch.uint8, device="cuda")
    off = torch.empty(dims[0] * dims[1] + 1, dtype=torch.int64, device="cuda")
    b.sparse_encode(rec, out, off)
    out_a, off_a = torch.empty_like(out), torch.empty_like(off)
    a.sparse_encode(rec, out_a, off_a)
    a.stats(); b.stats()
    assert (off.cpu() == off_a.cpu()).all()
    n = int(off[-1])
    assert (out[:n].cpu() == out_a[:n].cpu()).all()
    a.close(); b.close()


def test_forget_when_the_buffer_is_reused():
    """ctx `a` aggregates job 1 into rec; ctx `b` then aggregates job 2 into the SAME buffer.  Without argus_forget
    `a` would still take rec for its own table and read job 1's sum plane; after it, `a` reads the records."""
    from paper_2606_20374_b200 import argus as A
    ev1, dims = _events("tiny")
    ev2, dims2 = _events("tiny", seed=777)
    assert dims == dims2 and not (ev1 == ev2).all()
    a, b = A.Argus(*dims), A.Argus(*dims)
    rec = a.alloc_records()
    _aggregate(a, ev1, rec)
    _, _, od1 = run_oracle(ev1, *dims)
    _same(_diag(a, rec), od1)
    _aggregate(b, ev2, rec)                      # the buffer now holds job 2
    _, _, od2 = run_oracle(ev2, *dims)
    _same(_diag(b, rec), od2)
    a.forget()
    _same(_diag(a, rec), od2)
    # a forgotten ctx owns no table: its accumulation calls refuse until the next reset
    for fn, args in ((a.aggregate, (None, 0, rec)), (a.phase_times, (rec,)), (a.pack_planes, (rec, 0, 1, None, None, dims[0], 0))):
        with pytest.raises(A.ArgusError) as e:
            fn(*args)
        assert e.value.code == A.ESTATE
    _aggregate(a, ev1, rec)                      # reset makes it the owner again
    _same(_diag(a, rec), od1)
    a.close(); b.close()
