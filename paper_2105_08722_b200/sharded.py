"""One catalogue on several GPUs: primaries sharded across ranks, one small collective.

The paper's only parallel loop is the one over primaries (OpenMP, per-thread copies of zeta summed at the end,
PAPER.md:487, :547).  Here every rank (one process per GPU, torch.distributed) holds the whole catalogue (<= 51 MB)
and calls encore_compute_shard with its own rank: the library evaluates eq. 34's sum over that rank's contiguous
range of cell-sorted primaries.  The only exchange on the data path is the sum of the partial zeta vectors
(<= 114 kB each): an all-gather followed by a sum in RANK ORDER on every rank, so that all ranks hold bit-identical
results (an all-reduce may add in a different order on different ranks or runs).  All arithmetic of the estimator
is in the CUDA library; this module only marshals the collective.
"""
from __future__ import annotations


def combine_partials(partial, group=None):
    """All-gather `partial` (any shape, same on all ranks) and add the pieces in rank order 0, 1, ..., W-1.

    Works on the backend of the process group (NCCL for CUDA tensors, gloo for CPU tensors in the tests)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return partial.clone()
    world = dist.get_world_size(group)
    pieces = [torch.empty_like(partial) for _ in range(world)]
    dist.all_gather(pieces, partial.contiguous(), group=group)
    total = pieces[0].clone()
    for r in range(1, world):
        total += pieces[r]          # fixed order: identical bits on every rank
    return total


def compute_sharded(plan, positions, weights=None, group=None, stream=None):
    """zeta of one catalogue with the primaries split over the ranks of `group`; returns the full zeta on every rank."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        rank, world = dist.get_rank(group), dist.get_world_size(group)
    else:
        rank, world = 0, 1
    partial = plan.compute_shard(positions, weights, rank, world, stream=stream)
    return combine_partials(partial, group)
