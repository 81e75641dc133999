"""Host-side partition of a batch of spectra over ranks.

Spectra are independent units in the sum-of-chi2 form (DESIGN.md C.2-3), so the path shards by contiguous
spectrum ranges with NO collective on the data path: every rank builds its own lasp_ctx (the emulator
table, grid and basis tables are replicated, <= 3.3 MB) and fits its slice.  torch.distributed is used
only for the barrier and the max-over-ranks time of bench.py.
"""
from __future__ import annotations


def shard_range(B: int, rank: int, world: int) -> tuple[int, int]:
    """[start, stop) of rank's contiguous slice; sizes differ by at most one, earlier ranks get the extra."""
    if world < 1 or not (0 <= rank < world) or B < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(B, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """The slowest rank's time (what bench.py reports); `dist` is an initialised torch.distributed or None."""
    if dist is None or not dist.is_initialized():
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
