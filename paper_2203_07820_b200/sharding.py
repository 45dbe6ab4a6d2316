"""Host-side helpers for the band-parallel (over vectors) multi-GPU layout.

Columns of the vector block are independent under the filter (Eq. 37 acts on every column separately), so
N GPUs = N replicas of the operator, each filtering its own columns: there is NO data-path collective.  The
only communication is the benchmark's barrier and the max-over-ranks of the measured time.
"""
from __future__ import annotations


def column_shard(n_columns: int, world: int, rank: int, multiple: int = 1):
    """Half-open column range [j0, j1) owned by `rank` when `n_columns` are split over `world` ranks in
    contiguous pieces whose sizes are multiples of `multiple` (except possibly the last non-empty one)."""
    if world < 1 or not (0 <= rank < world) or n_columns < 0 or multiple < 1:
        raise ValueError("bad shard arguments")
    units = (n_columns + multiple - 1) // multiple
    base, extra = divmod(units, world)
    u0 = rank * base + min(rank, extra)
    u1 = u0 + base + (1 if rank < extra else 0)
    return min(u0 * multiple, n_columns), min(u1 * multiple, n_columns)


def aggregate_max(value: float, world: int) -> float:
    """max over ranks of a host scalar (device timing of the slowest rank); identity for world == 1."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
