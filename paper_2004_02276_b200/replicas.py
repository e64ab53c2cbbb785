"""N > 1 GPUs: the hot path does not shard (one GPU, no domain decomposition, no collectives --
BASELINE.json north_star), so `bench.py --gpus N` runs N independent replicas, one per rank.
The only cross-rank traffic is the barrier and the max-over-ranks of the timed region."""


def world():
    import torch.distributed as dist
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def max_over_ranks(seconds: float, device=None) -> float:
    """Slowest rank's time (all-reduce MAX); identity for a single process."""
    import torch
    import torch.distributed as dist
    if world() == 1:
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(points_per_rank: int, steps: int, seconds_local: float, device=None) -> float:
    """Whole-job grid-point updates/s: all ranks' points x steps over the slowest rank's time."""
    return world() * points_per_rank * steps / max_over_ranks(seconds_local, device)
