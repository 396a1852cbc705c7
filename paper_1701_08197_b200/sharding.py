"""Multi-GPU plumbing for the LOF path: streams (subbands, baselines, beams) are independent units
(PAPER.md:89 "different frequency subbands are processed on different compute nodes", :178), so N GPUs
take contiguous ranges of streams and no data-path collective exists.  Only the benchmark timing is
reduced across ranks (max of the per-rank device time)."""


def stream_range(rank, world, n_streams):
    """Contiguous [lo, hi) of streams owned by `rank`; sizes differ by at most one; every stream is
    owned exactly once; a rank's history rings live with its streams."""
    if not (0 <= rank < world) or n_streams < 0:
        raise ValueError("bad rank/world/n_streams")
    base, rem = divmod(n_streams, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value, device=None):
    """Max of a python float over all ranks of the default process group (identity without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank, steps, max_ms, world):
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return world * units_per_rank * steps / (max_ms * 1e-3)
