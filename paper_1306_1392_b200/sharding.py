"""Multi-GPU plumbing: slices are independent ("a given reconstructed line depends on
one and only one sinogram"), so the stack is partitioned over ranks and there is NO data-path
collective.  The only communication is the max-over-ranks of the measured time in bench.py.
"""
from __future__ import annotations

from typing import Optional, Tuple


def slice_range(n_slices: int, world_size: int, rank: int) -> Tuple[int, int]:
    """[first, last) slices of `rank`: contiguous, sizes differ by at most one, covers every slice once."""
    if world_size <= 0 or not (0 <= rank < world_size) or n_slices < 0:
        raise ValueError("bad partition request")
    base, rem = divmod(n_slices, world_size)
    first = rank * base + min(rank, rem)
    return first, first + base + (1 if rank < rem else 0)


def max_over_ranks(value: float, dist=None) -> float:
    """MAX all-reduce of a scalar over the default process group (gloo: CPU tensor, nccl: CUDA)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_slices(local, n_slices: int, dist=None):
    """Rank 0 gets the full stack [n_slices, ...] assembled from every rank's slice_range block (used by
    tests and by callers that want one array; the reconstruction itself never needs it)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local
    import torch
    world, rank = dist.get_world_size(), dist.get_rank()
    spans = [slice_range(n_slices, world, r) for r in range(world)]
    most = max(b - a for a, b in spans)
    # collectives want equal shapes: pad every block to the largest one, trim after the gather
    padded = torch.zeros((most,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    padded[: local.shape[0]] = local
    bufs = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(bufs, padded)
    if rank != 0:
        return None
    return torch.cat([buf[: b - a] for buf, (a, b) in zip(bufs, spans)], dim=0)
