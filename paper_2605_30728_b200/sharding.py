"""Multi-GPU host logic: the path shards by ids with no exchange step.

Each rank owns a contiguous slice of the batch, its own handle (packed store + metadata replica) and its own PCIe link.
A collective is needed only if a consumer wants the whole batch on every rank (one all-gather of the decoded slices).
Nothing here touches the row data; it is index arithmetic plus thin torch.distributed calls.
"""
from __future__ import annotations

import numpy as np


def shard_bounds(n: int, rank: int, world: int):
    """Contiguous slice [lo, hi) of a batch of n ids for `rank`; sizes differ by at most one; covers [0, n) exactly."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_ids(ids: np.ndarray, rank: int, world: int) -> np.ndarray:
    lo, hi = shard_bounds(len(ids), rank, world)
    return ids[lo:hi]


def max_over_ranks(value: float, device=None) -> float:
    """Device/CPU max-reduction of a per-rank time (multi-GPU numbers are the max over ranks)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_gather_rows(local_rows, n_total: int, world: int):
    """All-gather of decoded row slices (shape [n_local, row_bytes]) into [n_total, row_bytes] on every rank.
    Slices are the shard_bounds slices, so ranks may differ by one row: pad to the largest, gather, trim."""
    import torch
    import torch.distributed as dist
    row_bytes = local_rows.shape[1]
    sizes = [shard_bounds(n_total, r, world)[1] - shard_bounds(n_total, r, world)[0] for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros((pad, row_bytes), dtype=local_rows.dtype, device=local_rows.device)
    buf[: local_rows.shape[0]] = local_rows
    outs = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(outs, buf)
    return torch.cat([o[:s] for o, s in zip(outs, sizes)], dim=0)
