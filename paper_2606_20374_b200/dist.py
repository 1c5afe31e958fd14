"""Multi-GPU plumbing: one process per GPU, torch.distributed for the barrier and
the max-over-ranks timing only.  The hot path partitions into independent jobs (a job = one table
of R ranks x T steps), so ranks share no data-path collective; bench.py reports weak scaling."""
from __future__ import annotations

import dataclasses
import os
from typing import Optional

import torch
import torch.distributed as dist


@dataclasses.dataclass
class World:
    rank: int = 0
    size: int = 1
    local_rank: int = 0
    backend: Optional[str] = None


def init_world(n_gpus: int, backend: Optional[str] = None) -> World:
    """Join the process group torchrun set up (RANK / WORLD_SIZE / MASTER_* in the environment).
    A plain `python bench.py` run (no WORLD_SIZE) is a world of one and needs no group."""
    size = int(os.environ.get("WORLD_SIZE", "1"))
    if n_gpus not in (0, size):
        raise RuntimeError(f"--gpus {n_gpus} but WORLD_SIZE={size}: launch one rank per GPU (torchrun)")
    if size == 1:
        return World()
    rank = int(os.environ["RANK"])
    local_rank = int(os.environ.get("LOCAL_RANK", rank))
    backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
    if backend == "nccl":
        torch.cuda.set_device(local_rank)
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=size)
    return World(rank, size, local_rank, backend)


def _dev(w: World):
    return torch.device("cuda", w.local_rank) if w.backend == "nccl" else torch.device("cpu")


def barrier(w: World) -> None:
    if w.size > 1:
        dist.barrier()


def max_over_ranks(w: World, value: float) -> float:
    """Device-timed durations are combined as the max over ranks (never wall clock)."""
    if w.size == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_dev(w))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(w: World, value: float) -> float:
    if w.size == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_dev(w))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_seed(base_seed: int, w: World) -> int:
    """Weak scaling: every GPU aggregates and diagnoses its own job of the named size, generated
    from its own seed (rank 0 keeps the N=1 bytes)."""
    return base_seed + 1000003 * w.rank


def finish(w: World) -> None:
    if w.size > 1 and dist.is_initialized():
        dist.destroy_process_group()
