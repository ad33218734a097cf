"""Sink sharding across ranks: the paper's scatter-compute-gather
 with one process per GPU.  Sinks are cut into contiguous blocks, one per rank; the
source stream is replicated.  The one real exchange step of the path is the all-gather of the
Newtonian accelerations between the Newton and the gradient sweep (Eq. 27 needs a_j of every
source).  No reduction is involved, so results are bit-identical to one GPU.

Pair sharding (`pair_sharded_acc_grad`) is the multi-GPU form of the pair-symmetric sweeps
(csrc/frost_sym.cu, frost_set_shard): every rank evaluates 1/world of the TILE PAIRS and produces
partial sums for all particles, which one all-reduce (sum) per sweep combines -- 24 B per particle
against ~N^2/world pair evaluations.

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


def _staged_through_host(t: torch.Tensor) -> bool:
    """gloo moves host memory: a CUDA tensor is exchanged through a host copy (the backend used to run
    several ranks on ONE device, bench.py --backend gloo --same-device; NCCL exchanges device memory)."""
    return t.is_cuda and dist.get_backend() == "gloo"


def all_gather_planes(local: torch.Tensor, n: int, rank: int, world: int,
                      out: torch.Tensor) -> torch.Tensor:
    """Assemble out[:, 0:n] from every rank's block out[:, lo:hi]; `local` is this rank's (3, hi-lo)."""
    if world == 1:
        lo, hi = shard_range(n, rank, world)
        out[:, lo:hi] = local
        return out
    sizes = [shard_range(n, r, world) for r in range(world)]
    blk = max(hi - lo for lo, hi in sizes)
    dev = torch.device("cpu") if _staged_through_host(local) else local.device
    send = torch.zeros((3, blk), dtype=local.dtype, device=dev)
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


def all_reduce_planes(t: torch.Tensor, world: int) -> torch.Tensor:
    """Sum the partial planes of all ranks in place (NCCL on GPUs, gloo in the CPU test)."""
    if world > 1:
        if _staged_through_host(t):
            h = t.cpu()
            dist.all_reduce(h, op=dist.ReduceOp.SUM)
            t.copy_(h)
        else:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def pair_sharded_acc_grad(world: int, acc_fn: Callable, grad_fn: Callable, acc: torch.Tensor,
                          grad: torch.Tensor):
    """One full acc+gradient pass with the pairs sharded over ranks.

    acc_fn(acc)        must write this rank's PARTIAL Eq. 24 sums for every particle into acc;
    grad_fn(acc, grad) must write this rank's PARTIAL Eq. 27 sums into grad, reading the complete acc.
    After the call acc and grad hold the complete sums on every rank."""
    acc_fn(acc)
    all_reduce_planes(acc, world)
    grad_fn(acc, grad)
    all_reduce_planes(grad, world)
