"""Multi-process plumbing for `bench.py --gpus N`: replicas only, no data-path collective.

Every rank simulates an independent replicate (own seed) of the same landscape; the job-level numbers are the
sum of the units processed and the max of the device times over ranks. Works with NCCL (GPU tensors) and with
gloo (CPU tensors; the world-size-2 test in tests/test_dist_gloo.py).
"""
import torch
import torch.distributed as dist


def replica_seed(seed, rank):
    """Seed of rank `rank`'s replicate simulation (distinct u64 per rank, rank 0 keeps the config's seed)."""
    return (int(seed) + int(rank)) & (2**64 - 1)


def aggregate(times_ms, units, device="cpu"):
    """times_ms, units: lists of per-rank floats. Returns (max over ranks of each time, sum over ranks of each unit)."""
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    u = torch.tensor(list(units), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return t.tolist(), u.tolist()


def throughput(units_total, time_ms_max):
    """Whole-job units per second: everything all ranks processed over the slowest rank's time."""
    return units_total / (time_ms_max * 1e-3)
