"""Replicas-only multi-GPU plumbing: every rank runs an independent simulation;
the only cross-rank traffic is the reduction of the timing and of the processed-unit counts.  No
data-path collective exists.  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU
tests)."""
import torch
import torch.distributed as dist


def reduce_replicas(ms_local, units_local, device="cpu"):
    """(max over ranks of ms_local, sum over ranks of units_local); identity when not distributed."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    n = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), float(n.item())


def replica_seed(seed, rank):
    """rank r simulates its own discharge"""
    return int(seed) + int(rank)


def throughput(units_total, steps, ms_max):
    """whole-job particle-steps per second"""
    return units_total * steps / (ms_max * 1e-3)
