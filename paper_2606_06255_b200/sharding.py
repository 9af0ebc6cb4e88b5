"""Multi-GPU plumbing: replicas only.

The M iterations of one cloud are strictly sequential and each ends in a global argmax
(PAPER.md:126), so one cloud is never split across GPUs; clouds are independent units.  With N
ranks every rank runs its own batch (weak scaling: per-GPU work fixed) or a slice of one batch;
there is NO data-path collective.  torch.distributed is used only for the barrier and the
max-over-ranks of the measured time.
"""
from __future__ import annotations


def shard_range(B: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slice [lo, hi) of B clouds owned by ``rank`` (sizes differ by at most one)."""
    if world < 1 or not (0 <= rank < world) or B < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(B, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def rank_seed(base_seed: int, rank: int, B: int) -> int:
    """Weak scaling: rank r draws clouds with seeds base + r*B .. base + r*B + B-1 (disjoint)."""
    return base_seed + rank * B


def max_over_ranks(value: float, dist=None) -> float:
    """MAX all-reduce of a Python float (gloo or nccl); identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return value
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
