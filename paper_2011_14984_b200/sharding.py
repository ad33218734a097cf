"""Sink sharding across ranks: the paper's scatter-compute-gather
 with one process per GPU.  Sinks are cut into contiguous blocks, one per rank; the
source stream is replicated.  The one real exchange step of the path is the all-gather of the
Newtonian accelerations between the Newton and the gradient sweep (Eq. 27 needs a_j of every
source).  No reduction is involved, so results are bit-identical to one GPU.

The compute is injected as callables so that the host logic can be exercised on CPU with gloo
(tests/test_sharding_gloo.py); on GPUs the callables are Frost.forces.
"""
from __future__ import annotations

from typing import Callable, Tuple

import torch
import torch.distributed as dist


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block [lo, hi) of rank `rank`: sizes differ by at most one, larger blocks first."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def all_gather_planes(local: torch.Tensor, n: int, rank: int, world: int,
                      out: torch.Tensor) -> torch.Tensor:
    """Assemble out[:, 0:n] from every rank's block out[:, lo:hi]; `local` is this rank's (3, hi-lo)."""
    if world == 1:
        lo, hi = shard_range(n, rank, world)
        out[:, lo:hi] = local
        return out
    sizes = [shard_range(n, r, world) for r in range(world)]
    blk = max(hi - lo for lo, hi in sizes)
    send = torch.zeros((3, blk), dtype=local.dtype, device=local.device)
    send[:, : local.shape[1]] = local
    recv = [torch.empty_like(send) for _ in range(world)]
    dist.all_gather(recv, send)
    for r, (lo, hi) in enumerate(sizes):
        out[:, lo:hi] = recv[r][:, : hi - lo]
    return out


def sharded_acc_grad(n: int, rank: int, world: int, acc_fn: Callable, grad_fn: Callable,
                     acc: torch.Tensor, grad: torch.Tensor):
    """One full acc+gradient pass with sinks sharded over ranks.

    acc_fn(sink_idx, acc)  must fill acc[:, sink_idx] with Eq. 24 sums over all sources;
    grad_fn(sink_idx, acc, grad) must fill grad[:, sink_idx] with Eq. 27 sums using the full acc.
    Returns this rank's (lo, hi)."""
    lo, hi = shard_range(n, rank, world)
    sink_idx = torch.arange(lo, hi, dtype=torch.int32, device=acc.device)
    acc_fn(sink_idx, acc)
    all_gather_planes(acc[:, lo:hi].contiguous(), n, rank, world, acc)
    grad_fn(sink_idx, acc, grad)
    return lo, hi
