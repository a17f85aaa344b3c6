"""Multi-GPU plumbing: the batch axis shards, nothing else does.

Every environment is independent ("all B environments are still processed simultaneously at
every node"), so N ranks evaluate N disjoint contiguous ranges of the batch with a replicated model and NO
data-path collective.  ``torch.distributed`` is used only for the barrier and the max-over-ranks of timings.
"""
from __future__ import annotations


def shard_range(B: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) of the batch axis owned by ``rank``: every shard but the last holds ceil(B / world) rounded
    up to a multiple of 4 environments (keeps every SoA row slice 16-byte aligned); the last takes what is left, and
    trailing ranks can be EMPTY when B is small (B = 10, world = 4: 4, 4, 2, 0) -- an empty shard is a legal B = 0 call."""
    if world <= 1:
        return 0, B
    q = -(-B // world)
    q = -(-q // 4) * 4
    lo = min(B, rank * q)
    hi = min(B, lo + q)
    return lo, hi


def soa_slice(a, lo: int, hi: int):
    """Slice the batch (last) axis of an SoA array / tensor; contiguous per row, a copy is needed to make the
    shard a dense [rows, hi - lo] buffer for one device."""
    return a[..., lo:hi]


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (timings are reported as the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
