"""Multi-GPU use of the sweep: independent replicas only.

The labeling step is global ("This problem of multi-cluster flip Monte Carlo is not a local one",
PAPER.md:70), so the path does not shard without an exchange step; on an 8-GPU box the ranks run
independent Markov chains (different seeds / temperatures) and no data-path collective exists.
The only cross-rank arithmetic is the benchmark's own bookkeeping below: the sum of the units all
ranks processed divided by the slowest rank's time.  Works on any torch.distributed backend
(NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Distinct Philox key per rank, so the replicas are independent chains."""
    return int(base_seed) + int(rank)


def aggregate_throughput(local_units: float, local_seconds: float, device=None):
    """(total units over all ranks, max seconds over ranks, units per second) -- collective call."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_units), float(local_seconds), float(local_units) / float(local_seconds)
    units = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    secs = torch.tensor([float(local_seconds)], dtype=torch.float64, device=device)
    dist.all_reduce(units, op=dist.ReduceOp.SUM)
    dist.all_reduce(secs, op=dist.ReduceOp.MAX)
    return float(units.item()), float(secs.item()), float(units.item()) / float(secs.item())
