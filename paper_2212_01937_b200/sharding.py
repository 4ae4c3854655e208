"""Multi-GPU plumbing (torch.distributed only; no arithmetic of the method).

The path shards over redshifts with every cosmology on every rank: forward values and grad_z stay
local; the per-cosmology sums (grad_params [4][S], logL [S]) need ONE all-reduce.  Works with any backend (nccl on GPUs,
gloo in the CPU tests).
"""
from __future__ import annotations


def shard_bounds(n: int, world: int, rank: int):
    """contiguous, balanced [lo, hi) of rank's redshift shard; the first n % world ranks get one extra element"""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allreduce_sums(*tensors):
    """in-place sum of the per-cosmology reductions over all ranks (no-op without an initialised process group)"""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return tensors
    for t in tensors:
        if t is not None:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return tensors
