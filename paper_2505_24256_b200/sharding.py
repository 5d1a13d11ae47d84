"""Host-side multi-GPU plumbing ("the coefficients can be distributed among
different GPUs").  The functions of a batch are independent, so the path shards by functions with NO
data-path collective: every rank calls the C-ABI on its own block of functions.  The only communication is
the timing reduction of bench.py (max over ranks) and, if the caller wants the results in one place, a gather
of the output columns.  Nothing here does modular arithmetic; it runs on CPU tensors too (gloo tests).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class Shard:
    rank: int
    world: int
    f_lo: int  # functions [f_lo, f_hi) of the global batch
    f_hi: int
    term_lo: int  # their terms [term_lo, term_hi) = columns of vals / out, rows of exps
    term_hi: int
    offsets: np.ndarray  # local int64 [f_hi - f_lo + 1], starting at 0


def shard_functions(offsets, world: int, rank: int) -> Shard:
    """Block partition of the F functions of a batch over `world` ranks, balanced by the solve's cost
    sum_f t_f^2 (the hot loop is quadratic in t): cut points are the prefix-cost quantiles.  Every rank gets
    a contiguous range (possibly empty when F < world)."""
    o = np.asarray(offsets, dtype=np.int64)
    F = len(o) - 1
    if world <= 0 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    t = np.diff(o).astype(np.float64)
    cost = np.concatenate([[0.0], np.cumsum(t * t)])
    cuts = [0]
    for r in range(1, world):
        target = cost[-1] * r / world
        f = int(np.searchsorted(cost, target, side="left"))
        if f > 0 and abs(cost[f - 1] - target) <= abs(cost[min(f, F)] - target):
            f -= 1
        cuts.append(min(max(f, cuts[-1]), F))
    cuts.append(F)
    f_lo, f_hi = cuts[rank], cuts[rank + 1]
    return Shard(rank, world, f_lo, f_hi, int(o[f_lo]), int(o[f_hi]), (o[f_lo:f_hi + 1] - o[f_lo]).copy())


def rank_seed_shift(rank: int) -> int:
    """Weak scaling (bench.py): rank r lifts its own batch of the same shape, seed = base + 1000 r."""
    return 1000 * int(rank)


def max_over_ranks(value: float, device="cpu") -> float:
    """Timing rule of the bench contract: a multi-GPU time is the MAX over ranks."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    tt = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def gather_columns(local_out, shard: Shard, T_tot: int):
    """Optional result collection: every rank contributes out[:, term_lo:term_hi]; returns the full
    [B, T_tot] tensor on every rank (all_gather of padded blocks; not on the timed path)."""
    import torch
    import torch.distributed as dist

    B = local_out.shape[0]
    world = dist.get_world_size()
    spans = [None] * world
    dist.all_gather_object(spans, (shard.term_lo, shard.term_hi))
    width = max(b - a for a, b in spans)
    pad = torch.zeros((B, max(width, 1)), dtype=local_out.dtype, device=local_out.device)
    pad[:, : local_out.shape[1]] = local_out
    blocks = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(blocks, pad)
    full = torch.empty((B, T_tot), dtype=local_out.dtype, device=local_out.device)
    for (a, b), blk in zip(spans, blocks):
        full[:, a:b] = blk[:, : b - a]
    return full
