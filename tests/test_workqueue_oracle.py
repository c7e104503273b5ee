"""Pins for the pure-Python workqueue oracle (oracle/workqueue_oracle.py).

P7 Table 4 arithmetic   P8 "split 14"
P9 brute-force enumeration of the rectangular grid + coverage invariants
"""
import os

import numpy as np
import pytest

from oracle import workqueue_oracle as wq

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(path):
    with open(os.path.join(GOLDEN, path)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def test_p7_table4_counters():
    """8 long rows (>= 16K tokens, so T >= 512 >> S), Hkv=8, G=4, d=128, 28 SMs: the printed
    'Decode CTA work/SM' and 'Merge MB' cells follow from tasks = B*Hkv*S and (d+2)*4 bytes per
    (task, query head) -- which is what pins the FP32 (m, l, acc[d]) partial format (A11, A14)."""
    seq = [16384 + 977 * i for i in range(8)]
    for engine, S, launches, work_per_sm, useful_mb, merge_mb, merge_launches in _rows("table4_counters.txt"):
        S = int(S)
        q = wq.build_workqueue(seq, 8, wq.Policy(tile_tokens=32, num_splits=S))
        assert q.num_tasks == 8 * 8 * S
        assert round(wq.cta_work_per_sm(q.num_tasks, 28), 1) == float(work_per_sm)
        mb = wq.merge_bytes(q.num_tasks, 4, 128) / 2 ** 20
        assert f"{mb:.2f}" == merge_mb
        if engine == "workqueue":
            assert q.decode_launches + q.merge_launches == int(float(launches))     # 2.00
            assert q.merge_launches == int(float(merge_launches))                   # 1.00
        # 'Useful KV MB' is sum(N_i) * 4096 B in MiB: 550.5 MiB is a whole number of tokens
        assert (float(useful_mb) * 2 ** 20) % 4096 == 0
    assert wq.useful_kv_bytes([10, 20], 8, 128) == 30 * 4096


def test_p8_auto_split_default():
    for sms, B, Hkv, split in _rows("auto_split.txt"):
        assert wq.auto_num_splits(int(B), int(Hkv), int(sms)) == int(split)
        pol = wq.Policy(num_splits=0, num_sms=int(sms))
        assert wq.build_workqueue([32768] * int(B), int(Hkv), pol).num_splits == int(split)
    assert wq.auto_num_splits(1, 8, 148) == 74
    assert wq.auto_num_splits(128, 8, 148) == 1
    assert wq.auto_num_splits(1, 1, 10 ** 6) == wq.AUTO_S_MAX


def _check_invariants(seq, Hkv, pol, q):
    B = len(seq)
    assert q.num_tasks == len(q.tasks)
    assert len(q.split_offsets) == B + 1 and q.split_offsets[0] == 0
    per = {}
    for idx, (i, g, s, tb, te) in enumerate(q.tasks):
        assert 0 <= i < B and 0 <= g < Hkv
        per.setdefault((i, g), []).append((s, tb, te, idx))
    for i in range(B):
        n_i = q.split_offsets[i + 1] - q.split_offsets[i]
        T = -(-int(seq[i]) // pol.tile_tokens)
        for g in range(Hkv):
            lst = per.get((i, g), [])
            assert len(lst) == n_i
            pos = 0
            for k, (s, tb, te, idx) in enumerate(lst):
                assert s == k
                # slot formula (A8): contiguous run per (row, kvh), canonical order
                assert idx == q.split_offsets[i] * Hkv + g * n_i + s
                if pol.route == wq.ROUTE_WORKQUEUE:
                    assert tb < te
                assert tb == pos or (tb >= te and tb == T)
                pos = max(pos, te)
            assert pos == T                      # tiles [0, T) covered exactly once, in order
    assert q.tasks == sorted(q.tasks, key=lambda t: (t[0], t[1], t[2]))


@pytest.mark.parametrize("mode", [wq.SPLIT_FIXED_COUNT, wq.SPLIT_FIXED_CHUNK])
def test_p9_bruteforce_and_invariants_fuzz(mode):
    rng = np.random.Generator(np.random.PCG64(1234 + mode))
    for trial in range(300):
        B = int(rng.integers(1, 9))
        Hkv = int(rng.choice([1, 4, 8]))
        tile = int(rng.choice([16, 32, 64, 128]))
        seq = [int(x) for x in rng.choice([0, 1, 15, 16, 17, 31, 32, 33, 100, 1000, 5000, 40000], size=B)]
        seq = [max(0, n + int(rng.integers(-3, 4))) for n in seq]
        S = int(rng.integers(1, 70))
        pol = wq.Policy(tile_tokens=tile, split_mode=mode, num_splits=S,
                        chunk_tiles=int(rng.integers(1, 40)))
        q = wq.build_workqueue(seq, Hkv, pol)
        assert q.tasks == wq.brute_force_tasks(seq, Hkv, pol)
        _check_invariants(seq, Hkv, pol, q)
        assert q.empty_ctas == 0
        # the rectangular route holds the same non-empty tasks plus the empty ones
        polr = wq.Policy(tile_tokens=tile, split_mode=mode, num_splits=S, chunk_tiles=pol.chunk_tiles,
                         route=wq.ROUTE_RECT)
        r = wq.build_workqueue(seq, Hkv, polr)
        assert r.num_tasks == B * Hkv * S
        assert [t for t in r.tasks if t[3] < t[4]] == q.tasks
        assert r.empty_ctas == r.num_tasks - q.num_tasks
        _check_invariants(seq, Hkv, polr, r)


def test_balanced_policy_bruteforce_invariants_and_closed_forms():
    """Reading A21 (BALANCED): the chunk search against an exhaustive scan over every c (the
    brute force tests the single-wave conditions in rationals), the coverage invariants, the
    single-wave guarantee (at most U (row, split) pairs, none longer than the chunk) and a few
    cases worked by hand."""
    rng = np.random.Generator(np.random.PCG64(77))
    for trial in range(400):
        B = int(rng.integers(1, 40))
        Hkv = int(rng.choice([4, 8]))
        tile = int(rng.choice([16, 32, 64]))
        U = int(rng.choice([4, 28, 148]))
        seq = [int(x) for x in rng.choice([0, 1, 16, 17, 100, 500, 1000, 5000, 40000, 65536], size=B)]
        seq = [max(0, n + int(rng.integers(-3, 4))) for n in seq]
        pol = wq.Policy(tile_tokens=tile, split_mode=wq.SPLIT_BALANCED, num_splits=int(rng.choice([0, 0, 7, 64])),
                        num_sms=U)
        q = wq.build_workqueue(seq, Hkv, pol)
        assert q.tasks == wq.brute_force_tasks(seq, Hkv, pol)
        _check_invariants(seq, Hkv, pol, q)
        T = [-(-n // tile) for n in seq if n > 0]
        W = sum(T)
        if W == 0:
            continue
        c2 = max(-(-256 // tile), -(-W // (32 * U)))
        assert all(te - tb <= max(q.chunk_tiles, -(-max(T) // q.num_splits)) for (_, _, _, tb, te) in q.tasks)
        if q.chunk_tiles != c2 or sum(-(-t // c2) for t in T) <= U:
            if pol.num_splits == 0:       # single wave (no cap on n_i in the way)
                assert q.split_offsets[-1] <= U
                assert -(-W // U) <= q.chunk_tiles <= -(-W // U) + c2
                # minimality: one tile less per pair would need more than U pairs (or undercut the mean)
                c = q.chunk_tiles - 1
                assert c < -(-W // U) or sum(-(-t // c) for t in T) > U
    # by hand, U = 148: one row of 32768 tokens, 32-token tiles: W = 1024, ceil(W/U) = 7,
    # ceil(1024/7) = 147 <= 148 -> chunk 7, 147 splits (146 of 7 tiles, one of 2)
    q = wq.build_workqueue([32768], 8, wq.Policy(tile_tokens=32, split_mode=wq.SPLIT_BALANCED, num_splits=0, num_sms=148))
    assert q.chunk_tiles == 7 and q.split_offsets == [0, 147] and q.tasks[146] == (0, 0, 146, 1022, 1024)
    # W <= U: every tile is its own task
    q = wq.build_workqueue([256], 8, wq.Policy(tile_tokens=32, split_mode=wq.SPLIT_BALANCED, num_splits=0, num_sms=148))
    assert q.chunk_tiles == 1 and q.split_offsets == [0, 8]
    # more rows than SMs: no single wave exists -> many-wave chunk max(8, ceil(W / (32 U)))
    q = wq.build_workqueue([3200] * 10, 8, wq.Policy(tile_tokens=32, split_mode=wq.SPLIT_BALANCED, num_splits=0, num_sms=4))
    assert q.chunk_tiles == 8 and q.split_offsets[-1] == 10 * 13          # T = 100 -> S_i = 13, c = 8, n = 13
    q = wq.build_workqueue([32000] * 10, 8, wq.Policy(tile_tokens=32, split_mode=wq.SPLIT_BALANCED, num_splits=0, num_sms=4))
    assert q.chunk_tiles == -(-10000 // 128)                              # W = 10000, 32 U = 128 -> 79


def test_known_small_case_by_hand():
    """N=100, tile 32 -> T=4; S=3 -> c=2, n=2: splits [0,2) and [2,4); N=10 -> T=1, n=1."""
    q = wq.build_workqueue([100, 10, 0], 2, wq.Policy(tile_tokens=32, num_splits=3))
    assert q.split_offsets == [0, 2, 3, 3]
    assert q.tasks == [(0, 0, 0, 0, 2), (0, 0, 1, 2, 4), (0, 1, 0, 0, 2), (0, 1, 1, 2, 4),
                       (1, 0, 0, 0, 1), (1, 1, 0, 0, 1)]
    assert (q.decode_launches, q.merge_launches) == (1, 1)
    # single split everywhere -> no merge launch; fused merge -> no merge launch
    assert wq.build_workqueue([100, 10], 2, wq.Policy(num_splits=1)).merge_launches == 0
    assert wq.build_workqueue([100, 10], 2, wq.Policy(num_splits=3, merge_mode=wq.MERGE_FUSED)).merge_launches == 0
    assert wq.build_workqueue([0, 0], 2, wq.Policy(num_splits=3)).decode_launches == 0
    # FIXED_CHUNK: uniform task size, n_i proportional to length, capped
    q = wq.build_workqueue([32 * 10, 32 * 3], 1, wq.Policy(tile_tokens=32, split_mode=wq.SPLIT_FIXED_CHUNK,
                                                           num_splits=4, chunk_tiles=2))
    # row 0: T=10, S_i=min(4,5)=4, c=3, n=4 ; row 1: T=3, S_i=min(4,2)=2, c=2, n=2
    assert q.split_offsets == [0, 4, 6]
    assert q.tasks == [(0, 0, 0, 0, 3), (0, 0, 1, 3, 6), (0, 0, 2, 6, 9), (0, 0, 3, 9, 10),
                       (1, 0, 0, 0, 2), (1, 0, 1, 2, 3)]


def test_algorithmic_bytes_definition():
    """K+V of the active rows + q in/out + table entries used + seq_lens."""
    b = wq.algorithmic_bytes([32768], B=1, Hq=32, Hkv=8, d=128, page_size=16)
    assert b == 32768 * 4096 + 2 * 32 * 128 * 2 + 2048 * 4 + 4
