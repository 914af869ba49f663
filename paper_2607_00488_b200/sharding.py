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


def shard_pad(P, world):
    """Length every rank's slice is padded to for the gather (the largest shard)."""
    return -(-int(P) // int(world))


def gather_shards(out_local, pad, gathered, P, world):
    """Strong scaling's only exchange, 8 P bytes per scan: every rank's out[lo:hi) -> the whole scan's out[P] on every
    rank.  `pad` [shard_pad] and `gathered` [world * shard_pad] are caller-owned buffers on out_local's device (no
    allocation per step); returns a tensor of P values in scan order (a fresh one unless the shards are equal-sized,
    where it is a view of `gathered`)."""
    import torch
    import torch.distributed as dist
    n = out_local.numel()
    pad[:n].copy_(out_local)
    dist.all_gather_into_tensor(gathered, pad) if gathered.is_cuda else dist.all_gather(
        list(gathered.view(world, -1).unbind(0)), pad)
    sp = pad.numel()
    if P == world * sp:
        return gathered
    return torch.cat([gathered[r * sp: r * sp + (shard_range(P, r, world)[1] - shard_range(P, r, world)[0])]
                      for r in range(world)])


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
