"""Host-side bookkeeping for running the path on N GPUs (one process per GPU).

The path shards by row (and by KV head) with NO data-path collective (DESIGN.md "Multi-GPU",
SURVEY.md sec. 8(e)): every rank decodes its own rows with its own page pool.  What is left for
`torch.distributed` is plumbing: which rows / which seeded trace a rank owns, a barrier around
the timed region, the MAX over ranks of the device time, and the whole-job aggregate.  The same
functions run on `gloo` (CPU tests, world_size 2) and on `nccl` (bench.py under torchrun).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def rank_seed(base_seed: int, rank: int) -> int:
    """Weak scaling: rank r replays its own seeded trace (replica r of the workload)."""
    return int(base_seed) + int(rank)


def shard_rows(B: int, world: int, rank: int) -> Tuple[int, int]:
    """Strong scaling by row: rows [lo, hi) of a batch of B rows belong to `rank`; contiguous,
    sizes differ by at most one, every row belongs to exactly one rank."""
    if world <= 0 or not (0 <= rank < world) or B < 0:
        raise ValueError("bad (B, world, rank) = (%d, %d, %d)" % (B, world, rank))
    base, rem = divmod(B, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(values: Sequence[float], device=None) -> List[float]:
    """Element-wise MAX over ranks of a few timings (all_reduce; identity when not initialised)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def sum_over_ranks(values: Sequence[int], device=None) -> List[int]:
    """Element-wise SUM over ranks of a few integer counts (rows decoded, launches)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([int(v) for v in values], dtype=torch.int64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [int(x) for x in t.cpu()]


def whole_job_tokens_per_s(rows_all_ranks: int, steps: int, ms_max: float) -> float:
    """Decode tokens/s of the whole job: one token per row per step, all ranks'
    rows, over the slowest rank's device time."""
    return rows_all_ranks * steps / (ms_max * 1e-3)
