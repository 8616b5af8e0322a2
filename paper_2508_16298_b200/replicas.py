"""Multi-GPU mode of the hot path: REPLICAS ONLY.

The paper runs on one GPU and the path has no exchange step worth sharding at these sizes
(SURVEY.md 8e), so N GPUs run N independent lattices (independent Markov chains / random vectors), one process
per GPU, with no data-path collective.  This module holds the host logic only: which seed a rank uses and how
per-rank timings and work counts are combined (max time over ranks, summed work), over any torch.distributed
backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

SEED_STRIDE = 1000


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank's lattice: rank 0 keeps the BASELINE config's seed, the others get disjoint streams."""
    assert rank >= 0
    return int(base_seed) + SEED_STRIDE * int(rank)


def aggregate(seconds_local: float, units_local: int, world: int):
    """-> (max over ranks of the local time, sum over ranks of the local work units)."""
    if world <= 1:
        return float(seconds_local), int(units_local)
    import torch
    import torch.distributed as dist
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([float(seconds_local)], dtype=torch.float64, device=dev)
    u = torch.tensor([int(units_local)], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())
