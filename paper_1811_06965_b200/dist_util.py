"""Rank plumbing for bench.py: barrier and max-over-ranks of a device time.  The GPipe path has no
data-path collective (BASELINE.json: "no sharding across GPUs and no collectives"); N > 1 runs are
independent replicas and torch.distributed only synchronises the timed region."""
from __future__ import annotations


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def barrier(world: int) -> None:
    d = _dist()
    if world > 1 and d is not None:
        d.barrier()


def max_over_ranks(value_ms: float, world: int) -> float:
    """Every rank gets the maximum of `value_ms` over all ranks."""
    d = _dist()
    if world <= 1 or d is None:
        return float(value_ms)
    import torch
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value_ms)], dtype=torch.float64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(units_per_rank: float, steps: int, max_ms: float, world: int) -> float:
    """value = units all ranks processed / the slowest rank's time (weak scaling, replicas)."""
    return units_per_rank * world * steps / (max_ms / 1e3)
