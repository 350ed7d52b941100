"""Host-side logic of the N > 1 ("replicas only") mode: every rank steps an independent replica of the
workload on its own GPU; there is no data-path collective.  What the ranks share is the timing protocol: a barrier on
both sides of the timed region, the MAX of the per-rank device times, and the whole-job aggregate.  torch.distributed
is the plumbing (nccl on GPUs, gloo in the CPU test)."""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of the ensemble member a rank steps (rank 0 keeps the configuration's own seed)."""
    return int(base_seed) + 1000 * int(rank)


def barrier(dist=None, sync=None):
    """Device synchronise (if given) + process-group barrier + device synchronise."""
    if sync is not None:
        sync()
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
        if sync is not None:
            sync()


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX over ranks of a per-rank scalar (the job is as slow as its slowest replica)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(cells_per_replica: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job cell-updates/s: all replicas' cells over the slowest replica's time."""
    return float(world) * float(cells_per_replica) * float(steps) / (float(ms_max) * 1e-3)
