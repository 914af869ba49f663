"""Multi-GPU plumbing: the path shards over parameter points (one theta never depends on another,
PAPER.md:202), so every rank owns a batch of points and a replica of the tables; there is no
data-path collective.  torch.distributed is used only for the barrier and the max-over-ranks of
the timed region (bench.py)."""
import numpy as np

from . import workloads as wl


def rank_points(name, rank):
    """Rank 0 folds the config's own scan; every further rank an independent seeded draw of the same
    shape and kinds (weak scaling: per-GPU work is fixed as the job grows)."""
    params, kinds = wl.scan_points(name)
    if rank > 0:
        params, kinds = wl.random_points(params.shape[0], kinds, seed=100003 * rank + 7)
    return np.ascontiguousarray(params), kinds


def shard_range(P, rank, world):
    """Contiguous slice [lo, hi) of P points owned by `rank` (strong-scaling split of one scan):
    sizes differ by at most one, every point is owned exactly once."""
    base, rem = divmod(int(P), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(x, device, world):
    """max of a python float over all ranks (device-timed durations are combined this way)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, points_per_rank, steps, ms):
    """evals/s of the whole job: all ranks' points over the slowest rank's time."""
    return world * points_per_rank * steps / (ms * 1e-3)
