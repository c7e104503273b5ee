"""Split-bound policy and compact workqueue -- pure-Python integer oracle.
TEST INFRASTRUCTURE, NOT THE PRODUCT (shares no code with the C++/CUDA builders).

Follows PAPER.md:63-67 (§3.3 row-local bounds: tile count, split range and final-tile size come
from N_i* = seq_lens[i]) and PAPER.md:71-75 (§3.4: for each active row i, KV head g and row-local
split s emit (row, kvh, split, t_begin, t_end) only if the tile interval is non-empty; partials
live in the compact slot range described by split_offsets).  Readings of what the paper leaves
open: A5 tile_tokens is a policy field, A6 ceil-chunk division of a row's tiles,
A7 canonical order row, kvh, split, A8 split_offsets = exclusive prefix sum of n_i,
A9 N_i = 0 rows emit nothing, A12 auto split count, A13 launch counting, A14 counter units,
A21 BALANCED: the chunk of a FIXED_CHUNK policy derived from the whole batch's true lengths
("CTA-work and length-based tile bounds"; per-row split counts are the paper's
future work).

Pins (tests/test_workqueue_oracle.py): brute-force enumeration of the rectangular grid,
coverage invariants, and the printed cells of Table 4 and §4.2's
"split 14".
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Sequence, Tuple

SPLIT_FIXED_COUNT = 0
SPLIT_FIXED_CHUNK = 1
SPLIT_BALANCED = 2
ROUTE_RECT = 0
ROUTE_WORKQUEUE = 1
MERGE_SEPARATE = 0
MERGE_FUSED = 1

AUTO_C_MIN = 4          # PAPER.md:85 "C_min = 4 CTAs/SM"
AUTO_S_MAX = 256
BAL_WAVES = 32          # A21: many-wave regime, about 32 (row, split) pairs per SM ...
BAL_MIN_TOKENS = 256    # ... of at least 256 tokens each


def ceil_div(a: int, b: int) -> int:
    return -(-a // b)


@dataclass(frozen=True)
class Policy:
    tile_tokens: int = 32                 # PAPER.md:50 "32-token tiles"
    split_mode: int = SPLIT_FIXED_COUNT
    num_splits: int = 1                   # FIXED_COUNT: S (0 = auto); FIXED_CHUNK: cap on n_i
    chunk_tiles: int = 0                  # FIXED_CHUNK: tiles per task (BALANCED: ignored)
    route: int = ROUTE_WORKQUEUE
    merge_mode: int = MERGE_SEPARATE
    num_sms: int = 0                      # only used by the auto rule and by BALANCED


def auto_num_splits(B: int, Hkv: int, num_sms: int) -> int:
    """Reading A12: S = clamp(ceil(C_min * SMs / (B * Hkv)), 1, 256).
    Pin: 28 SMs, B=1, Hkv=8 -> 14 ("selects split 14")."""
    return max(1, min(AUTO_S_MAX, ceil_div(AUTO_C_MIN * num_sms, max(1, B * Hkv))))


def resolve_num_splits(policy: Policy, B: int, Hkv: int) -> int:
    if policy.num_splits > 0:
        return policy.num_splits
    if policy.split_mode != SPLIT_FIXED_COUNT:
        return AUTO_S_MAX
    assert policy.num_sms > 0, "auto split needs num_sms"
    return auto_num_splits(B, Hkv, policy.num_sms)


def balanced_chunk(seq_lens: Sequence[int], policy: Policy) -> int:
    """Reading A21 (include/pkv.h BALANCED).  U = num_sms, T_i = ceil(N_i / tile_tokens),
    W = sum_i T_i.  Many waves: c2 = max(ceil(256 / tile_tokens), ceil(W / (32 U))).  Single wave:
    the smallest c with ceil(W/U) <= c <= ceil(W/U) + c2 and sum_i ceil(T_i / c) <= U (at most
    one (row, split) pair per SM; the busiest SM's share c exceeds the mean by at most one
    many-wave chunk).  The chunk is that c if it exists, else c2."""
    U = policy.num_sms
    assert U > 0, "BALANCED needs num_sms"
    T = [ceil_div(int(N), policy.tile_tokens) for N in seq_lens if int(N) > 0]
    W = sum(T)
    if W == 0:
        return 1
    c2 = max(ceil_div(BAL_MIN_TOKENS, policy.tile_tokens), ceil_div(W, BAL_WAVES * U))
    for c in range(ceil_div(W, U), ceil_div(W, U) + c2 + 1):
        if sum(ceil_div(t, c) for t in T) <= U:
            return c
    return c2


def row_splits(N: int, policy: Policy, S: int, chunk: int = 0) -> Tuple[int, int, int]:
    """(T, c, n) for one row: tile count, tiles per split, number of non-empty splits.
    `chunk`: the batch-wide chunk of a BALANCED policy (balanced_chunk)."""
    T = ceil_div(N, policy.tile_tokens) if N > 0 else 0
    if T == 0:
        return 0, 0, 0
    if policy.split_mode == SPLIT_FIXED_COUNT:
        S_i = S
    elif policy.split_mode == SPLIT_BALANCED:
        S_i = min(S, ceil_div(T, chunk))
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
    chunk_tiles: int = 0                          # FIXED_CHUNK / BALANCED: resolved tiles per task


def build_workqueue(seq_lens: Sequence[int], Hkv: int, policy: Policy) -> WorkQueue:
    """The algorithm of SURVEY.md §8(c) C2, step by step."""
    B = len(seq_lens)
    S = resolve_num_splits(policy, B, Hkv)
    tasks: List[Tuple[int, int, int, int, int]] = []
    offsets = [0]
    max_n = 0
    nonempty = 0
    chunk = 0
    if policy.split_mode == SPLIT_BALANCED:
        chunk = balanced_chunk(seq_lens, policy)
    elif policy.split_mode == SPLIT_FIXED_CHUNK:
        chunk = policy.chunk_tiles
    for i in range(B):
        T, c, n = row_splits(int(seq_lens[i]), policy, S, chunk)
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
                     grid_ctas=num_tasks, empty_ctas=num_tasks - nonempty, chunk_tiles=chunk)


def brute_force_tasks(seq_lens: Sequence[int], Hkv: int, policy: Policy):
    """Independent restatement used to pin build_workqueue (pin P9): enumerate every (i, g, s) of
    a rectangular grid wide enough for any row, compute its tile interval directly from the
    row's own (T, c) and keep the non-empty ones."""
    B = len(seq_lens)
    S = resolve_num_splits(policy, B, Hkv)
    out = []
    chunk = policy.chunk_tiles
    if policy.split_mode == SPLIT_BALANCED:
        # exhaustive: every c from 1 up, the single-wave conditions tested as stated (in
        # rationals: mean = W/U <= c, and c < mean + c2 + 1 i.e. c <= ceil(mean) + c2), first
        # hit wins; else the many-wave chunk
        from fractions import Fraction
        U = policy.num_sms
        Ts = [(int(N) + policy.tile_tokens - 1) // policy.tile_tokens for N in seq_lens if int(N) > 0]
        W = sum(Ts)
        if W == 0:
            chunk = 1
        else:
            mean = Fraction(W, U)
            c2 = max(-(-BAL_MIN_TOKENS // policy.tile_tokens), -(-W // (BAL_WAVES * U)))
            chunk = c2
            for c in range(1, max(Ts) + c2 + 2):
                pairs = sum((t + c - 1) // c for t in Ts)
                if pairs <= U and mean <= c and c - c2 - 1 < mean:
                    chunk = c
                    break
    for i in range(B):
        N = int(seq_lens[i])
        T = (N + policy.tile_tokens - 1) // policy.tile_tokens
        if T == 0:
            continue
        if policy.split_mode == SPLIT_FIXED_COUNT:
            S_i = S
        else:
            S_i = min(S, (T + chunk - 1) // chunk)
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
