"""World-size-2 gloo tests of the multi-process plumbing bench.py uses (CPU only)."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2606_20374_b200 import dist as D
    w = D.init_world(world, backend="gloo")
    D.barrier(w)
    mx = D.max_over_ranks(w, 10.0 + rank)          # slowest rank decides the time
    sm = D.sum_over_ranks(w, 100.0 * (rank + 1))   # whole-job units
    seed = D.job_seed(1234, w)
    D.finish(w)
    q.put((rank, w.size, mx, sm, seed))


def test_world_of_two_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    assert all(r[1] == 2 for r in res)
    assert all(r[2] == 11.0 for r in res)          # max over ranks
    assert all(r[3] == 300.0 for r in res)         # sum over ranks
    assert res[0][4] == 1234 and res[1][4] != 1234  # rank 0 keeps the N=1 bytes; others get their own job


def test_world_of_one_needs_no_group(monkeypatch):
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    from paper_2606_20374_b200 import dist as D
    w = D.init_world(1)
    assert (w.rank, w.size) == (0, 1)
    assert D.max_over_ranks(w, 3.5) == 3.5 and D.sum_over_ranks(w, 2.0) == 2.0
    D.barrier(w)


def test_shards_are_independent_jobs():
    """Different job seeds give different event bytes of the same shape (weak scaling)."""
    import dataclasses
    import numpy as np
    from paper_2606_20374_b200 import dist as D
    from paper_2606_20374_b200.workload import build_workload, scaled
    spec = scaled("tiny", n_ranks=2, n_steps=1, n_events=300)
    a = build_workload(spec).expand_host()
    b = build_workload(dataclasses.replace(spec, seed=D.job_seed(spec.seed, D.World(1, 2, 1, "gloo")))).expand_host()
    assert a.shape == b.shape and (a["rank"] == b["rank"]).all()
    assert not (a["end_ns"] == b["end_ns"]).all()


def test_reference_arm_runs_on_cpu():
    """bench.py --impl reference times the oracle on the host; rank > 0 exits without work."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ)
    env.pop("RANK", None)
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--workload",
                        "tiny", "--steps", "2", "--warmup", "1"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0
    env["RANK"] = "1"
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--workload",
                        "tiny", "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""


# ---- the exchange of a rank-sharded job: layout only, no method arithmetic ---------------
def _exchange_worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import numpy as np
    from paper_2606_20374_b200 import dist as D
    from paper_2606_20374_b200 import sharded as Sh
    w = D.init_world(world, backend="gloo")
    R, T, S, P = 7, 3, 5, 2
    lay = Sh.Layout(world, R, T, S, P)
    # a known whole-job sum table x[r][t][s] and span table y[r][t][k]; every rank builds its own slice
    x = (np.arange(R * T * S, dtype=np.int64).reshape(R, T, S) * 1000003) % 99991
    y = (np.arange(R * T * (P + 1), dtype=np.int64).reshape(R, T, P + 1) * 7919) % 10007
    r0, r1 = lay.ranks[rank]
    # what argus_pack_planes writes for an all-to-all: for d: [T][S_d][R_g], then the span part [T][P+1][R_g]
    send = np.concatenate([x[r0:r1, :, s0:s1].transpose(1, 2, 0).reshape(-1) for s0, s1 in lay.sigs])
    span_part = y[r0:r1].transpose(1, 2, 0).reshape(-1)
    sig_plane, span_plane = Sh.exchange_all_to_all(lay, rank, torch.from_numpy(send.copy()),
                                                   torch.from_numpy(span_part.copy()))
    s0, s1 = lay.sigs[rank]
    ok_sig = np.array_equal(sig_plane.numpy().reshape(T, s1 - s0, R), x[:, :, s0:s1].transpose(1, 2, 0))
    ok_span = np.array_equal(span_plane.numpy().reshape(T, P + 1, R), y.transpose(1, 2, 0))
    D.finish(w)
    q.put((rank, ok_sig, ok_span, lay.send_counts(rank), lay.recv_counts(rank)))


def test_sharded_exchange_layout_world_of_two_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_exchange_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(r[1] and r[2] for r in res), res
    # 7 ranks -> 4 + 3; 5 sigs -> 3 + 2; T = 3: rank 0 sends 3*3*4 and 3*2*4 elements
    assert res[0][3] == [36, 24] and res[1][3] == [27, 18]
    assert res[0][4] == [36, 27] and res[1][4] == [24, 18]


def test_sharded_split_is_balanced_and_contiguous():
    from paper_2606_20374_b200.sharded import Layout, split
    assert split(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert split(2, 4) == [(0, 1), (1, 2), (2, 2), (2, 2)]
    lay = Layout(8, 4096, 1, 4096, 16)
    assert all(b - a == 512 for a, b in lay.ranks) and sum(lay.send_counts(3)) == 512 * 4096
    assert 8 * sum(sum(lay.send_counts(g)) for g in range(8)) == 8 * 4096 * 4096      # 134 MB in total
