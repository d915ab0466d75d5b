"""Batch partition for multi-GPU runs: spectra are independent, so ranks take contiguous slices of the
batch and exchange nothing.  Host logic only (no CUDA), covered by the world_size-2 gloo test."""
from __future__ import annotations


def shard_bounds(batch: int, world_size: int, rank: int):
    """Contiguous slice [lo, hi) of `batch` spectra for `rank`; sizes differ by at most one; empty slices allowed."""
    if batch < 0 or world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad shard arguments")
    base, rem = divmod(batch, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks_ms(local_ms: float, dist=None) -> float:
    """Step time of the whole job = the slowest rank's device time (MAX all-reduce; identity without a process group)."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(local_ms)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None) -> float:
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
