"""Multi-GPU plumbing: IM columns are independent, so the mode axis shards
with no data-path collective.  One process per GPU; torch.distributed is used only for barriers,
max-over-ranks timing and, when a caller wants the replicated matrix, one all_gather of the
per-rank column blocks (contiguous because the IM is column-major)."""
from __future__ import annotations

from typing import Callable, List, Optional, Tuple


def partition_modes(n_modes: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous, balanced mode ranges [begin, end) per rank; the first n_modes % world ranks get
    one extra mode.  Ranks beyond n_modes get empty ranges."""
    if n_modes < 0 or world < 1:
        raise ValueError("n_modes >= 0 and world >= 1 required")
    base, extra = divmod(n_modes, world)
    out, b = [], 0
    for r in range(world):
        e = b + base + (1 if r < extra else 0)
        out.append((b, e))
        b = e
    return out


def weak_scaling_plan(units_per_rank: int, world: int) -> dict:
    """Every rank processes its own workload of ``units_per_rank`` columns (independent problems)."""
    return {"scaling": "weak", "units_per_rank": int(units_per_rank), "world": int(world),
            "total_units": int(units_per_rank) * int(world)}


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (timings are reported as the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def sharded_columns(n_modes: int, compute: Callable[[int, int], "object"], gather: bool = False,
                    rank: Optional[int] = None, world: Optional[int] = None):
    """Run ``compute(begin, end)`` (-> tensor [end-begin][rows], i.e. a block of IM columns) on this
    rank's mode range.  With ``gather`` the blocks of all ranks are all_gathered into the replicated
    [n_modes][rows] matrix (uneven ranges are padded to the largest block for the collective)."""
    import torch
    import torch.distributed as dist
    if world is None:
        world = dist.get_world_size() if dist.is_initialized() else 1
    if rank is None:
        rank = dist.get_rank() if dist.is_initialized() else 0
    ranges = partition_modes(n_modes, world)
    b, e = ranges[rank]
    block = compute(b, e)
    if not gather or world == 1:
        return block, (b, e)
    rows = block.shape[1]
    biggest = max(r[1] - r[0] for r in ranges)
    padded = torch.zeros((biggest, rows), dtype=block.dtype, device=block.device)
    padded[: e - b] = block
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded)
    full = torch.cat([parts[r][: ranges[r][1] - ranges[r][0]] for r in range(world)], dim=0)
    return full, (b, e)
