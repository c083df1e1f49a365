"""Multi-GPU mode of the path: independent replicas only.

BASELINE.json's north_star scopes the hot path to one GPU with no collectives, so N GPUs run N
independent lattices (own seeds): weak scaling with no data-path collective.
The only cross-rank traffic is plumbing around the timed region -- agreeing on the lattice size,
the barrier, and the max-over-ranks of the device-timed duration -- which is what this module
holds, so that it can be tested on CPU with the gloo backend (tests/test_replicas.py).
"""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Seed of rank's replica: distinct Philox keys, rank 0 keeps the workload's own seed."""
    return int(base_seed) + 1000 * int(rank)


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def agree_min(value: int, device="cpu") -> int:
    """The smallest `value` over all ranks (every replica runs the same lattice size)."""
    dist = _dist()
    if dist is None or dist.get_world_size() == 1:
        return int(value)
    import torch
    t = torch.tensor([int(value)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return int(t.item())


def max_over_ranks(ms: float, device="cpu") -> float:
    """The slowest rank's duration: the time the whole job took."""
    dist = _dist()
    if dist is None or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier() -> None:
    dist = _dist()
    if dist is not None and dist.get_world_size() > 1:
        dist.barrier()


def job_rate(updates_per_rank: int, world: int, ms: float) -> float:
    """Whole-job spin updates/ns: all replicas' updates over the max-over-ranks time."""
    return world * updates_per_rank / (ms * 1e6)
