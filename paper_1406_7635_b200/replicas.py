"""Multi-GPU = independent replicas: the FFT convolution does not shard without two
all-to-alls of the whole spectrum per evaluation, and the paper is single-GPU, so
N GPUs run N independent simulations (parameter sweeps, the 3000-start search of L426). This module
holds the host-side logic only: which replica a rank runs and how per-rank timings become one
whole-job number. No data-path collective exists; the only communication is the timing reduction.
"""
import torch
import torch.distributed as dist


def replica_seed(base_seed, rank):
    """Seed of the replica a rank simulates: distinct per rank, reproducible."""
    return int(base_seed) + int(rank)


def shard_jobs(njobs, rank, world):
    """Indices of the independent jobs (e.g. sweep points) rank `rank` of `world` runs: round robin."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    return list(range(rank, njobs, world))


def max_over_ranks(value, device="cpu"):
    """Max of a per-rank float over all ranks (identity without an initialised process group)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device="cpu"):
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank, ms_this_rank, device="cpu"):
    """Whole-job throughput [units/s]: units all ranks processed / max-over-ranks time."""
    total = sum_over_ranks(units_this_rank, device)
    ms = max_over_ranks(ms_this_rank, device)
    return total / (ms * 1e-3), ms
