"""Multi-GPU bookkeeping: planes are independent (Algorithm 1 never lets two planes
interact, :136-146), so a job shards by contiguous plane ranges with the PSFs replicated and NO
data-path collective.  torch.distributed is used only to agree on a barrier and on the slowest
rank's time (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def plane_range(n_planes: int, rank: int, world: int) -> tuple[int, int]:
    """[p0, p1) of `rank`: contiguous, sizes differ by at most one pair, every range starts on an
    even plane so that the FFT engine's (2m, 2m+1) pairing is the same as in a single-rank run."""
    if n_planes < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("bad shard arguments")
    pairs = (n_planes + 1) // 2
    lo = (pairs * rank) // world
    hi = (pairs * (rank + 1)) // world
    return min(2 * lo, n_planes), min(2 * hi, n_planes)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of one scalar (the step time); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: list[int] | int, seconds_max: float, world: int = 1) -> float:
    """Whole-job units per second: everything all ranks processed / the slowest rank's time."""
    total = units_per_rank * world if isinstance(units_per_rank, int) else sum(units_per_rank)
    return total / seconds_max
