"""Multi-GPU plumbing (replicas only).  The particle step has no data-path collective: every
rank advances an independent replica of the workload (its own seed), and the ranks meet only to agree on the timing
of the job: the slowest rank's device time and the sum of the super-droplet steps all ranks processed."""
import torch
import torch.distributed as dist


def replica_seed(base_seed, rank):
    """Seed of the replica that rank `rank` advances (rank 0 keeps the base seed of the single-GPU run)."""
    return int(base_seed) + int(rank)


def job_totals(ms_local, units_local, device="cpu"):
    """(max over ranks of ms_local, sum over ranks of units_local); identity without an initialised process group.
    `device` is where the reduction tensors live: the rank's cuda device under NCCL, "cpu" under gloo."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def job_throughput(ms_local, units_local, device="cpu"):
    """Whole-job throughput in units per second: all ranks' units over the slowest rank's time."""
    ms, units = job_totals(ms_local, units_local, device)
    return units / (ms * 1e-3) if ms > 0 else 0.0
