"""Split-bound policy and compact workqueue -- pure-Python integer oracle.
TEST INFRASTRUCTURE, NOT THE PRODUCT (shares no code with the C++/CUDA builders).

Follows PAPER.md:63-67 (§3.3 row-local bounds: tile count, split range and final-tile size come
from N_i* = seq_lens[i]) and PAPER.md:71-75 (§3.4: for each active row i, KV head g and row-local
split s emit (row, kvh, split, t_begin, t_end) only if the tile interval is non-empty; partials
live in the compact slot range described by split_offsets).  Readings of what the paper leaves
open: A5 tile_tokens is a policy field, A6 ceil-chunk division of a row's tiles,
A7 canonical order row, kvh, split, A8 split_offsets = exclusive prefix sum of n_i,
A9 N_i = 0 rows emit nothing, A12 auto split count, A13 launch counting, A14 counter units.

Pins (tests/test_workqueue_oracle.py): brute-force enumeration of the rectangular grid,
coverage invariants, and the printed cells of Table 4 and §4.2's
"split 14".
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Sequence, Tuple

SPLIT_FIXED_COUNT = 0
SPLIT_FIXED_CHUNK = 1
ROUTE_RECT = 0
ROUTE_WORKQUEUE = 1
MERGE_SEPARATE = 0
MERGE_FUSED = 1

AUTO_C_MIN = 4          # PAPER.md:85 "C_min = 4 CTAs/SM"
AUTO_S_MAX = 256


def ceil_div(a: int, b: int) -> int:
    return -(-a // b)


@dataclass(frozen=True)
class Policy:
    tile_tokens: int = 32                 # PAPER.md:50 "32-token tiles"
    split_mode: int = SPLIT_FIXED_COUNT
    num_splits: int = 1                   # FIXED_COUNT: S (0 = auto); FIXED_CHUNK: cap on n_i
    chunk_tiles: int = 0                  # FIXED_CHUNK: tiles per task
    route: int = ROUTE_WORKQUEUE
    merge_mode: int = MERGE_SEPARATE
    num_sms: int = 0                      # only used by the auto rule


def auto_num_splits(B: int, Hkv: int, num_sms: int) -> int:
    """Reading A12: S = clamp(ceil(C_min * SMs / (B * Hkv)), 1, 256).
    Pin: 28 SMs, B=1, Hkv=8 -> 14 ("selects split 14")."""
    return max(1, min(AUTO_S_MAX, ceil_div(AUTO_C_MIN * num_sms, max(1, B * Hkv))))


def resolve_num_splits(policy: Policy, B: int, Hkv: int) -> int:
    if policy.num_splits > 0:
        return policy.num_splits
    if policy.split_mode == SPLIT_FIXED_CHUNK:
        return AUTO_S_MAX
    assert policy.num_sms > 0, "auto split needs num_sms"
    return auto_num_splits(B, Hkv, policy.num_sms)


def row_splits(N: int, policy: Policy, S: int) -> Tuple[int, int, int]:
    """(T, c, n) for one row: tile count, tiles per split, number of non-empty splits."""
    T = ceil_div(N, policy.tile_tokens) if N > 0 else 0
    if T == 0:
        return 0, 0, 0
    if policy.split_mode == SPLIT_FIXED_COUNT:
        S_i = S
    else:
        S_i = min(S, ceil_div(T, policy.chunk_tiles))
    c = ceil_div(T, S_i)
    n = ceil_div(T, c)
    return T, c, n


@dataclass
class WorkQueue:
    tasks: List[Tuple[int, int, int, int, int]]   # (row, kvh, split, t_begin, t_end)
    split_offsets: List[int]                      # [B+1]; slot(i,g,s) = split_offsets[i]*Hkv + g*n_i + s
    num_tasks: int
    num_splits: int                               # resolved S
    decode_launches: int
    merge_launches: int
    grid_ctas: int                                # CTAs a non-persistent launch would need
    empty_ctas: int                               # of which write neutral states (rect route only)


def build_workqueue(seq_lens: Sequence[int], Hkv: int, policy: Policy) -> WorkQueue:
    """The algorithm of SURVEY.md §8(c) C2, step by step."""
    B = len(seq_lens)
    S = resolve_num_splits(policy, B, Hkv)
    tasks: List[Tuple[int, int, int, int, int]] = []
    offsets = [0]
    max_n = 0
    nonempty = 0
    for i in range(B):
        T, c, n = row_splits(int(seq_lens[i]), policy, S)
        nonempty += n * Hkv
        max_n = max(max_n, n)
        if policy.route == ROUTE_WORKQUEUE:
            offsets.append(offsets[-1] + n)
            for g in range(Hkv):
                for s in range(n):
                    tasks.append((i, g, s, s * c, min((s + 1) * c, T)))
        else:
            # rectangular (B, Hkv, S) grid: every split has a CTA; empty ones carry an empty
            # interval t_begin = t_end = T and write the neutral state
            offsets.append(offsets[-1] + S)
            for g in range(Hkv):
                for s in range(S):
                    tb = min(s * c, T) if T > 0 else 0
                    te = min((s + 1) * c, T) if T > 0 else 0
                    tasks.append((i, g, s, tb, te))
    num_tasks = len(tasks)
    if policy.route == ROUTE_WORKQUEUE:
        slots_per_row_max = max_n
    else:
        slots_per_row_max = S if B > 0 else 0
    decode_launches = 1 if num_tasks > 0 else 0
    merge_launches = 0 if (slots_per_row_max <= 1 or policy.merge_mode == MERGE_FUSED
                           or num_tasks == 0) else 1
    return WorkQueue(tasks=tasks, split_offsets=offsets, num_tasks=num_tasks, num_splits=S,
                     decode_launches=decode_launches, merge_launches=merge_launches,
                     grid_ctas=num_tasks, empty_ctas=num_tasks - nonempty)


def brute_force_tasks(seq_lens: Sequence[int], Hkv: int, policy: Policy):
    """Independent restatement used to pin build_workqueue (pin P9): enumerate every (i, g, s) of
    a rectangular grid wide enough for any row, compute its tile interval directly from the
    row's own (T, c) and keep the non-empty ones."""
    B = len(seq_lens)
    S = resolve_num_splits(policy, B, Hkv)
    out = []
    for i in range(B):
        N = int(seq_lens[i])
        T = (N + policy.tile_tokens - 1) // policy.tile_tokens
        if T == 0:
            continue
        if policy.split_mode == SPLIT_FIXED_COUNT:
            S_i = S
        else:
            S_i = min(S, (T + policy.chunk_tiles - 1) // policy.chunk_tiles)
        c = (T + S_i - 1) // S_i
        for g in range(Hkv):
            for s in range(S_i):
                lo, hi = s * c, min((s + 1) * c, T)
                if lo < hi:
                    out.append((i, g, s, lo, hi))
    return out


# ---------------------------------------------------------------- Table 4 counters

def merge_bytes(num_slots: int, G: int, d: int) -> int:
    """Reading A14: one pass over the partial states, (d+2) FP32 words per (slot, query head)."""
    return num_slots * G * (d + 2) * 4


def useful_kv_bytes(seq_lens: Sequence[int], Hkv: int, d: int, elem_bytes: int = 2) -> int:
    """K+V bytes resident for the active rows ("Useful KV MB")."""
    return sum(int(n) for n in seq_lens) * 2 * Hkv * d * elem_bytes


def cta_work_per_sm(num_tasks: int, num_sms: int) -> float:
    """"Decode CTA work/SM" = tasks / #SMs (2048/28 = 73.1, 1280/28 = 45.7)."""
    return num_tasks / float(num_sms)


def algorithmic_bytes(seq_lens: Sequence[int], B: int, Hq: int, Hkv: int, d: int, page_size: int) -> int:
    """Roofline bytes of one decode step: K+V resident for the active rows,
    q in and out out, the block-table entries used and seq_lens."""
    kv = useful_kv_bytes(seq_lens, Hkv, d)
    qo = 2 * B * Hq * d * 2
    meta = sum(ceil_div(int(n), page_size) for n in seq_lens) * 4 + B * 4
    return kv + qo + meta
