"""Multi-GPU plumbing for bench.py.  The path shards by independent series: every rank
sweeps its own realisations of the workload, there is NO data-path collective, and the only communication is
the timing reduction (barrier + max over ranks).  Host logic only; runs under `gloo` on CPU in the tests."""
from __future__ import annotations

import os


def env_rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def realisations_for_rank(rank: int, world: int, per_rank: int = 1):
    """Weak scaling: rank r sweeps realisation indices [r*per_rank, (r+1)*per_rank) of the workload (distinct noise
    seeds), so per-GPU work is fixed as the job grows."""
    if not (0 <= rank < world):
        raise ValueError("rank outside world")
    return list(range(rank * per_rank, (rank + 1) * per_rank))


def init_process_group(backend: str):
    import torch.distributed as dist
    rank, world, _ = env_rank_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29512")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    """Every rank contributes its own device-timed duration; the job's time is the slowest rank's."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int, device="cpu") -> float:
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, ms_this_rank: float, world: int, device="cpu"):
    """value = units all ranks processed / max-over-ranks time.  Returns (units_per_second, max_ms)."""
    total = sum_over_ranks(units_this_rank, world, device)
    ms = max_over_ranks(ms_this_rank, world, device)
    return total / (ms * 1e-3), ms
