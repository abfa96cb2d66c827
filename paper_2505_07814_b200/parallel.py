"""Data-parallel sharding of a minibatch over ranks (one process per GPU).

Scan positions of a minibatch are independent units: each rank runs the fused
forward/adjoint kernels on its own contiguous shard of the positions with replicated object and
probe, and the only exchange is one sum all-reduce of the partial object / probe (/ global tilt)
gradients and the loss per minibatch -- NCCL over NVLink on GPUs (PAPER.md:199-201 does the same
through HF Accelerate).  Position gradients belong to the shard's own rows and are all-gathered.

The compute itself is passed in as a callable, so this host logic is also exercised on CPU with
the gloo backend (tests/test_parallel_gloo.py).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(B: int, rank: int, world: int):
    """Contiguous balanced split of range(B): the first B % world ranks get one extra position."""
    base, extra = divmod(B, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def _real_view(t: torch.Tensor) -> torch.Tensor:
    return torch.view_as_real(t) if t.is_complex() else t


def allreduce_sum(tensors, group=None):
    """In-place sum over ranks of every tensor (complex tensors through their real view)."""
    for t in tensors:
        if t is not None:
            dist.all_reduce(_real_view(t), op=dist.ReduceOp.SUM, group=group)


def sharded_gradient(compute, B: int, g_object, g_probe, g_positions, g_tilt_global=None, loss=None, group=None):
    """Run ``compute(lo, hi)`` on this rank's shard, then combine.

    ``compute(lo, hi)`` must fill g_object, g_probe, g_tilt_global and loss with the shard's
    partial sums and rows lo:hi of g_positions (other rows untouched).  On return every rank holds
    the full-minibatch gradients.
    """
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    lo, hi = shard_range(B, rank, world)
    g_positions.zero_()
    compute(lo, hi)
    allreduce_sum([g_object, g_probe, g_tilt_global, loss, g_positions], group=group)
    return lo, hi
