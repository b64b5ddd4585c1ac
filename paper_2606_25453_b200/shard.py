"""Host-side multi-rank plumbing: the hot path shards as INDEPENDENT problems, one
per rank, with no data-path collective.  Only the timing reduction (max over ranks) uses torch.distributed."""


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of the problem rank `rank` works on: same recipe, disjoint streams."""
    return int(base_seed) + 1000 * int(rank)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a per-rank time (ms); identity when torch.distributed is not initialised."""
    if dist is None or not dist.is_available() or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, world: int, ms_max: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time (units / s)."""
    return world * units_per_rank / (ms_max * 1e-3)
