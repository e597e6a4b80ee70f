"""Multi-GPU plumbing of bench.py: one process per GPU, every rank an independent lattice ("trivial
parallelization over disorder realizations" -- the path shards by independent units, so there is NO data-path
collective; only the timing and the final aggregation use torch.distributed).

Holds no arithmetic of the method.  Works with any backend: NCCL on the GPU box, gloo in the CPU tests.
"""
import os


def env_rank():
    """(rank, local_rank, world_size) as torchrun exports them; (0, 0, 1) for a plain `python bench.py`."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def rank_seed(base_seed, rank):
    """Seed of the lattice a rank owns: distinct per rank, so the N lattices are independent realisations."""
    return int(base_seed) + int(rank)


def max_over_ranks(value, dist=None, device="cpu"):
    """Largest `value` over all ranks (the timed region ends when the slowest rank is done)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, dist=None, device="cpu"):
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_flips_per_ns(updates_this_rank, ms_this_rank, dist=None, device="cpu"):
    """BASELINE metric over all ranks: (updates of every rank) / (slowest rank's time).  Weak scaling: each rank brings
    its own lattice, so the numerator grows with the world size."""
    total = sum_over_ranks(updates_this_rank, dist, device)
    ms = max_over_ranks(ms_this_rank, dist, device)
    return total / (ms * 1e6), ms
