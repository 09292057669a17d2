"""Multi-GPU plumbing of the benchmark: the path does not shard ("replicas only"), so
N ranks run N independent replicas and the only cross-rank traffic is the timing reduction.

Kept free of CUDA so that the rank logic is testable with the gloo backend on CPU.
"""
import os


def rank_info():
    """(rank, world_size, local_rank) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed(step, rank):
    """Seed of replica `rank` at timed step `step`: distinct streams per rank, reproducible."""
    return int(step) + 7919 * int(rank)


def reduce_stats(times_ms, units, device="cpu"):
    """Whole-job aggregate of per-rank measurements.

    times_ms: dict name -> elapsed milliseconds on this rank   (reduced with MAX: the job is as
              slow as its slowest rank)
    units:    dict name -> work units this rank processed      (reduced with SUM)
    Returns (times_max, units_sum) as plain dicts; identity when not under torch.distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return dict(times_ms), dict(units)
    tk, uk = sorted(times_ms), sorted(units)
    t = torch.tensor([float(times_ms[k]) for k in tk], dtype=torch.float64, device=device)
    u = torch.tensor([float(units[k]) for k in uk], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return ({k: t[i].item() for i, k in enumerate(tk)}, {k: u[i].item() for i, k in enumerate(uk)})


def throughput(units_sum, time_max_ms):
    """units per second of the whole job."""
    return units_sum / (time_max_ms * 1e-3)
