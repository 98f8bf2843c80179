"""Multi-GPU plumbing of the benchmark: the path shards over independent segments,
so ranks never exchange data; they only agree on who takes which segments and on the slowest time."""


def shard_segments(rank: int, world: int, batch_per_rank: int):
    """Weak scaling: rank r takes segments [r*batch, (r+1)*batch) of the seeded stream."""
    assert 0 <= rank < world and batch_per_rank >= 0
    first = rank * batch_per_rank
    return first, batch_per_rank


def max_over_ranks(values, device=None):
    """element-wise MAX of a list of floats over all ranks (identity when not distributed)"""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.tolist()]


def aggregate_throughput(world: int, batch_per_rank: int, n: int, ms_per_step: float) -> float:
    """whole-job input samples per second: the units all ranks processed / the slowest rank's time"""
    return world * batch_per_rank * n / (ms_per_step * 1e-3)
