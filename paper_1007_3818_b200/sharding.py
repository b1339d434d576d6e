"""Multi-GPU sharding of the hot path: patch groups are independent once their ghost shells
are filled (PAPER.md:13,35 — this is what lets the paper batch them to a GPU and decompose domains across MPI
ranks), so a batch is split into contiguous ranges of the group index, one per rank, and the step needs NO
collective. Only the timing of a multi-rank run is reduced (max over ranks). Host-side logic only; no CUDA."""
import torch
import torch.distributed as dist


def shard_range(n_groups: int, rank: int, world: int):
    """Contiguous, balanced partition: the first n_groups % world ranks get one extra group. Returns (start, stop)."""
    if world < 1 or not (0 <= rank < world) or n_groups < 0:
        raise ValueError("bad shard request: n_groups=%d rank=%d world=%d" % (n_groups, rank, world))
    base, extra = divmod(n_groups, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device=None) -> float:
    """max of a per-rank scalar (a time) over all ranks; identity when torch.distributed is not initialised."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: int, world: int, seconds_max: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return world * units_per_rank / seconds_max
