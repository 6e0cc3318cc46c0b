"""Multi-GPU host logic: the path has no exchange step (independent systems / replicas),
so ranks only agree on who builds which systems and on the timing (max over ranks)."""
import torch
import torch.distributed as dist


def shard_systems(n_systems: int, world: int, rank: int):
    """Contiguous, balanced slice [lo, hi) of the systems owned by `rank` (sizes differ by at most 1)."""
    base, rem = divmod(n_systems, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value: float, device="cpu") -> float:
    """Timing rule: a multi-rank number is the max over ranks."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu") -> float:
    """Whole-job throughput: all ranks' units / max-over-ranks time."""
    return sum_over_ranks(units_this_rank, device) / max_over_ranks(seconds_this_rank, device)
