"""Host-side logic of the N > 1 launch ("replicas only").

The graded path runs on one GPU and has no exchange step, so `bench.py --gpus N` advances N
independent replicas of the workload, one process per GPU, with no data-path collective.  What the
ranks share is bookkeeping only: a per-rank seed, the barrier around the timed region, the maximum
over ranks of the device time and the sum of the site updates.  This module holds that logic so that
it can be tested on CPU with the `gloo` backend (tests/test_replicas_gloo.py); it contains none of the
method's arithmetic.
"""
import torch
import torch.distributed as dist


def rank_seed(base_seed, rank):
    """Seed of rank `rank`'s replica: distinct droplet placements, same workload shape."""
    return int(base_seed) + 1000 * int(rank)


def max_over_ranks(value, device="cpu"):
    """Maximum of a float over all ranks (identity when torch.distributed is not initialised)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device="cpu"):
    """Sum of a float over all ranks (identity when torch.distributed is not initialised)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_mlups(sites_this_rank, steps, ms_this_rank, device="cpu"):
    """Whole-job MLUPS: all ranks' site updates over the slowest rank's device time.
    Returns (mlups, ms_max)."""
    ms = max_over_ranks(ms_this_rank, device)
    updates = sum_over_ranks(float(sites_this_rank) * float(steps), device)
    return updates / ms / 1e3, ms
