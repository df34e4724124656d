"""Multi-GPU plumbing.  The JUMP hot path of one box runs on one GPU (replicas only): N GPUs run
N independent replicas of the same system that differ in their Philox key only, with no data-path collective.  The only
communication is the timing reduction (max over ranks) of bench.py."""


def rank_seed(seed, rank):
    """Philox key of replica `rank`: the seed advanced by a large odd stride, so replica streams never coincide."""
    return (int(seed) + 0x9E3779B97F4A7C15 * int(rank)) & 0xFFFFFFFFFFFFFFFF


def max_over_ranks(value, dist=None, device=None):
    """MAX all-reduce of one float over the process group (identity without one)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(per_rank_units, elapsed_s, dist=None, device=None):
    """Whole-job throughput: units all ranks processed / max-over-ranks time."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(per_rank_units) / float(elapsed_s)
    import torch
    dev = device if device is not None else "cpu"
    u = torch.tensor([float(per_rank_units)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()) / max_over_ranks(elapsed_s, dist, device)
