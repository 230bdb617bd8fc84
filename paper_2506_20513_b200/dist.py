"""Shot sharding across ranks: shots are independent given the model, so each rank
sweeps its own contiguous block of shots and ONE all-reduce(sum) of the two gradient planes per
iteration completes the gradient; traces need no exchange.  Host logic only -- the kernels never
see another rank."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_shots(nshots: int, rank: int, world: int) -> range:
    """Contiguous, balanced block of shot indices for `rank` (the first nshots % world ranks get one more)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(nshots, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def allreduce_gradients(grad_eps_r: torch.Tensor, grad_sigma: torch.Tensor, group=None) -> None:
    """Sum the per-rank partial gradients in place (NCCL on GPUs, gloo in the CPU tests)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(grad_eps_r, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(grad_sigma, op=dist.ReduceOp.SUM, group=group)
