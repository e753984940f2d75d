"""Host-side logic of the N > 1 path: no arithmetic of the method.

The fused update shards along the WEIGHT with no collective: a rank that holds rows [r0, r1) of W
(and of m, v, the int8 scales) needs columns [r0, r1) of dY and the whole of X, and its result is
exactly the corresponding rows of the single-GPU result (tiles are independent, PAPER.md:273-279
Prop. 1; the shard's gradient is complete, Prop. 2(i)).  Data-parallel replicas do
NOT shard it (v is quadratic in G, Prop. 2(ii)).  The only cross-rank step is the timing
reduction bench.py uses (max over ranks).
"""
from __future__ import annotations

ROW_ALIGN = 128   # one tile row block; keeps every rank's shard tile-aligned


def shard_rows(out: int, world: int, rank: int, align: int = ROW_ALIGN) -> tuple[int, int]:
    """Rows [r0, r1) of W owned by `rank`: contiguous, `align`-aligned, sizes differ by <= align."""
    if not (0 <= rank < world):
        raise ValueError("rank outside world")
    blocks = (out + align - 1) // align
    base, extra = divmod(blocks, world)
    b0 = rank * base + min(rank, extra)
    b1 = b0 + base + (1 if rank < extra else 0)
    return min(out, b0 * align), min(out, b1 * align)


def shard_problem(d: dict, world: int, rank: int) -> dict | None:
    """Row shard of one problem dict (keys X, dY, W, m, v[, m_scale, v_scale]); None if empty.
    W/m/v/scales are row slices (views, updated in place); dY's column slice is a view too (the ABI takes its
    row pitch, include/forge.h lddy)."""
    out = d["W"].shape[0]
    r0, r1 = shard_rows(out, world, rank)
    if r1 <= r0:
        return None
    s = {"X": d["X"], "dY": d["dY"][:, r0:r1]}
    for k in ("W", "m", "v", "m_scale", "v_scale"):
        if d.get(k) is not None:
            s[k] = d[k][r0:r1]
    s["rows"] = (r0, r1)
    return s


def max_over_ranks(value: float, device=None) -> float:
    """The timing rule of bench.py: the slowest rank's device time."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
