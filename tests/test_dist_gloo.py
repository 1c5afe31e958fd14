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
