"""Multi-GPU plumbing: spins are independent and the only coupling is
the sum over spins per ADC sample (:194), so spins are partitioned contiguously across ranks, the plan is
replicated, and ONE collective adds the per-rank signals (n_adc complex fp32).  Final magnetisation and
PER_SPIN output stay sharded (no collective).  torch.distributed is plumbing only; nothing here computes
any of the method's arithmetic."""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when not launched by it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def shard_bounds(n_spins: int, rank: int, world_size: int):
    """Contiguous [lo, hi) of the spins owned by `rank`; sizes differ by at most one, every spin owned once."""
    if world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad rank / world_size")
    base, rem = divmod(int(n_spins), world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def reduce_signal(signal, group=None, deterministic=False):
    """In-place sum over ranks of a complex64 signal tensor [n_adc] (SUM_ALL output).  NCCL all-reduce on
    GPU tensors, gloo on CPU tensors; complex is reduced through its real view.  A no-op when
    torch.distributed is not initialised (single GPU).

    deterministic=True: all-gather the per-rank signals and add them in rank order on every rank, so the result
    does not depend on the collective's algorithm (ring / tree / in-switch reduction) -- the multi-GPU
    continuation of the fixed-order two-pass reduction inside one GPU; costs world_size x the
    bytes of the all-reduce, still <= 8 MB x world_size once per simulation."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return signal
    view = torch.view_as_real(signal) if signal.is_complex() else signal
    if not deterministic:
        dist.all_reduce(view, op=dist.ReduceOp.SUM, group=group)
        return signal
    world = dist.get_world_size(group)
    parts = [torch.empty_like(view) for _ in range(world)]
    dist.all_gather(parts, view.contiguous(), group=group)
    acc = parts[0].clone()
    for r in range(1, world):     # fixed order: ((s0 + s1) + s2) + ...
        acc += parts[r]
    view.copy_(acc)
    return signal
