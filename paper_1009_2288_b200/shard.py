"""Slice-sharded multi-GPU plumbing ("one slice per GPU").

The path shards trivially: slices are independent reconstructions, so rank r owns a contiguous block of
slices and there is NO collective on the data path. torch.distributed is used only to agree on timing
(max over ranks) and to gather small per-rank summaries. Works with the nccl backend (CUDA tensors, used by
bench.py) and with gloo (CPU tensors, used by the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def slice_range(rank: int, world: int, slices_per_rank: int) -> range:
    """Weak scaling: every rank reconstructs `slices_per_rank` slices; global slice ids are contiguous
    per rank, so the seeded inputs of a job are the same whatever the rank count of a given slice."""
    if not (0 <= rank < world) or slices_per_rank < 1:
        raise ValueError("slice_range: bad rank / world / slices_per_rank")
    return range(rank * slices_per_rank, (rank + 1) * slices_per_rank)


def split_slices(n_slices: int, world: int) -> list[range]:
    """Strong scaling: n_slices split into `world` contiguous, near-equal blocks (first ranks get the
    remainder)."""
    if world < 1 or n_slices < 0:
        raise ValueError("split_slices: bad arguments")
    base, extra = divmod(n_slices, world)
    out, start = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append(range(start, start + n))
        start += n
    return out


def max_over_ranks(values, device="cpu") -> list[float]:
    """Element-wise maximum of a short list of floats over all ranks (identity without a process group)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def job_throughput(units_per_rank: int, world: int, ms_per_rank: float, device="cpu") -> tuple[float, float]:
    """(whole-job units per second, max-over-ranks milliseconds): all ranks processed units_per_rank."""
    (ms,) = max_over_ranks([ms_per_rank], device)
    return world * units_per_rank / (ms * 1e-3), ms
