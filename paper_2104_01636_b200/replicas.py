"""Multi-GPU = independent replicas (replicas only).

BASELINE.json's north_star fixes the solver at one GPU with no domain decomposition and no
inter-GPU traffic, so `bench.py --gpus N` runs N independent solves, one process per GPU, each on
its own seeded workload (seed offset = rank).  The only communication is the timing protocol of
the bench contract: a barrier on both sides of the timed region and a max / sum over ranks of two
scalars.  No data-path collective exists and none is invented.
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass
class Rank:
    rank: int
    local_rank: int
    world: int
    backend: str | None      # None: single process, torch.distributed not initialised


def init(backend: str | None = None) -> Rank:
    """Read RANK/LOCAL_RANK/WORLD_SIZE (torchrun) and initialise torch.distributed if world > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1:
        return Rank(0, local, 1, None)
    import torch
    import torch.distributed as dist
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29511")
    if backend == "nccl":
        torch.cuda.set_device(local)
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Rank(rank, local, world, backend)


def seed_offset(r: Rank) -> int:
    """Replica r solves the config generated with seed + 1000*r (rank 0 = the config itself)."""
    return 1000 * r.rank


def _device(r: Rank):
    import torch
    return torch.device("cuda", r.local_rank) if r.backend == "nccl" else torch.device("cpu")


def barrier(r: Rank):
    if r.world > 1:
        import torch.distributed as dist
        if r.backend == "nccl":
            dist.barrier(device_ids=[r.local_rank])
        else:
            dist.barrier()


def reduce_scalars(r: Rank, values, op: str):
    """All-reduce a short list of floats with op in {'max', 'sum'}; identity when world == 1."""
    if r.world == 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return [float(v) for v in t.cpu().tolist()]


def aggregate_throughput(r: Rank, units_this_rank: float, seconds_this_rank: float):
    """Whole-job throughput: (sum of units over ranks) / (max of time over ranks)."""
    (units,) = reduce_scalars(r, [units_this_rank], "sum")
    (secs,) = reduce_scalars(r, [seconds_this_rank], "max")
    return units / secs, units, secs


def finalize(r: Rank):
    if r.world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
