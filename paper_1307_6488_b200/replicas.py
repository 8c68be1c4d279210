"""Multi-GPU plumbing of the benchmark: the path has no data-path collective ("replicas
only"), so N ranks run N independent replicas and only the timing is reduced: whole-job throughput =
(units all ranks processed) / (slowest rank's time).  Backend-agnostic (nccl on GPUs, gloo in the CPU tests)."""
import torch


def aggregate_throughput(local_seconds, units_per_rank, dist=None, device="cpu"):
    """Returns (whole_job_units_per_second, max_seconds_over_ranks).  `dist` is torch.distributed (initialised)
    or None for a single process."""
    t = torch.tensor([float(local_seconds)], dtype=torch.float64, device=device)
    world = 1
    if dist is not None and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        world = dist.get_world_size()
    worst = float(t.item())
    return world * units_per_rank / worst, worst


def replica_seed(base_seed, rank):
    """Every replica evolves its own seeded data."""
    return int(base_seed) + int(rank)
