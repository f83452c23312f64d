"""Multi-GPU plumbing: snapshots are independent ("no need for synchronisation
mechanisms"), so the path shards along time with NO data-path collective; torch.distributed is
used only for the barrier and the max-over-ranks timing reduction of the benchmark."""
from __future__ import annotations


def shard_time_steps(n_t: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous, balanced split of time steps [0, n_t) over ranks: returns (t0, t1) of `rank`.
    The first n_t % world ranks get one extra step; empty ranges are allowed (n_t < world)."""
    if world < 1 or not (0 <= rank < world) or n_t < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_t, world)
    t0 = rank * base + min(rank, extra)
    return t0, t0 + base + (1 if rank < extra else 0)


def barrier() -> None:
    """torch.distributed barrier (no-op when not initialised or world size 1)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, ms_this_rank: float, device=None) -> tuple[float, float]:
    """Whole-job throughput = units all ranks processed / max-over-ranks time; returns (units/s, ms)."""
    ms = max_over_ranks(ms_this_rank, device)
    units = sum_over_ranks(units_this_rank, device)
    return (units / (ms / 1e3) if ms > 0 else 0.0), ms
