"""Pins for oracle/route_oracle.py: the length-bucket route and the
calibrated cost model.

P11 Table 4's bucket row: 8 distinct lengths at split 32 -> 16.00 launches, 8.00 merge launches,
    2048 tasks = 73.1 per SM, 4.06 MB of merge state
P12 the cost of both Table-4 routes from the printed constants, worked out by hand below
P13 closed forms of the three terms; the occupancy factor on both sides of C_r = C_min
P14 gates and margins on constructed cases
"""
import os

import numpy as np
import pytest

from oracle import route_oracle as ro
from oracle import workqueue_oracle as wq

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(path):
    with open(os.path.join(GOLDEN, path)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


TABLE4 = {r[0]: r for r in _rows("table4_counters.txt")}
SEQ8 = [16384 + 977 * i for i in range(8)]           # 8 long rows, 8 distinct lengths


def test_p11_table4_bucket_row():
    engine, S, launches, work_per_sm, useful_mb, merge_mb, merge_launches = TABLE4["buckets"]
    pol = wq.Policy(tile_tokens=32, num_splits=int(S), route=wq.ROUTE_RECT)
    c, per_bucket = ro.bucket_route(SEQ8, 8, 4, 128, pol, bucket_tokens=1)
    assert c.buckets == 8 and [rows for rows, _ in per_bucket] == [[i] for i in range(8)]
    assert f"{c.launches:.2f}" == launches                                   # 16.00
    assert f"{c.merge_launches:.2f}" == merge_launches                       # 8.00
    assert c.tasks == 2048 and round(wq.cta_work_per_sm(c.tasks, 28), 1) == float(work_per_sm)   # 73.1
    assert f"{c.merge_bytes / 2 ** 20:.2f}" == merge_mb                      # 4.06
    assert c.empty_tasks == 0
    # the workqueue row through the same counters
    engine, S, launches, work_per_sm, useful_mb, merge_mb, merge_launches = TABLE4["workqueue"]
    w = ro.single_route(SEQ8, 8, 4, 128, wq.Policy(tile_tokens=32, num_splits=int(S)))
    assert (f"{w.launches:.2f}", f"{w.merge_launches:.2f}", f"{w.merge_bytes / 2 ** 20:.2f}") == (launches, merge_launches, merge_mb)
    assert round(wq.cta_work_per_sm(w.tasks, 28), 1) == float(work_per_sm)


def test_bucket_grouping_readings():
    lens = [5000, 0, 4999, 5000, 17, 4990, 32]
    assert ro.group_buckets(lens, 1) == [(17, [4]), (32, [6]), (4990, [5]), (4999, [2]), (5000, [0, 3])]
    assert ro.group_buckets(lens, 16) == [(32, [4, 6]), (4992, [5]), (5008, [0, 2, 3])]
    assert ro.group_buckets(lens, 8192) == [(8192, [0, 2, 3, 4, 5, 6])]       # one coarse masked bucket
    assert ro.group_buckets([0, 0], 1) == []
    # a single coarse bucket over the whole batch IS the rectangular route, empties included
    pol = wq.Policy(tile_tokens=32, num_splits=8, route=wq.ROUTE_RECT)
    active = [n for n in lens if n > 0]
    c, per = ro.bucket_route(lens, 8, 4, 128, pol, 8192)
    r = ro.single_route(active, 8, 4, 128, pol)
    assert (c.launches, c.tasks, c.empty_tasks, c.merge_bytes) == (r.launches, r.tasks, r.empty_tasks, r.merge_bytes)
    assert c.empty_tasks > 0 and per[0][0] == [0, 2, 3, 4, 5, 6]
    # exact buckets never pad: every row of a bucket has the same tile count, so with S <= T no empties
    c1, _ = ro.bucket_route([4096, 4096, 8192], 8, 4, 128, pol, 1)
    assert c1.buckets == 2 and c1.empty_tasks == 0 and c1.launches == 4


def test_p12_table4_route_costs_by_hand():
    """Table 4 + the constants of PAPER.md:85.  Useful KV = 550.5 MiB =
    577 241 088 B; beta = 331.2 GB/s = 331 200 B/us -> 577241088 / 331200 = 1742.877681... us, both
    routes are above C_min (73.1 and 45.7 >= 4), so the occupancy factor is 1.
      buckets:   16 * 8.19 = 131.04 us;  4.0625 MiB = 4 259 840 B / 331200 = 12.861836... us
      workqueue:  2 * 8.19 =  16.38 us;  2.5390625 MiB = 2 662 400 B / 331200 = 8.038647... us
    The 16-vs-2 launch case must prefer the workqueue."""
    beta, c_min, lam, sms = (float(x) for x in _rows("cost_model_constants.txt")[0][:4])
    k = ro.CostConstants(beta, lam, c_min, int(sms))
    assert k == ro.RTX3060
    kv = int(550.5 * 2 ** 20)
    assert kv == 577241088
    b = ro.route_cost(kv, int(4.0625 * 2 ** 20), 16, 2048, k)
    w = ro.route_cost(kv, int(2.5390625 * 2 ** 20), 2, 1280, k)
    assert b.stream_us == pytest.approx(1742.8776811594, rel=1e-12) and w.stream_us == b.stream_us
    assert b.launch_us == pytest.approx(131.04, rel=1e-12) and w.launch_us == pytest.approx(16.38, rel=1e-12)
    assert b.merge_us == pytest.approx(12.8618357488, rel=1e-11) and w.merge_us == pytest.approx(8.0386473430, rel=1e-11)
    assert b.total_us == pytest.approx(1886.7795169082, rel=1e-11)
    assert w.total_us == pytest.approx(1767.2963285024, rel=1e-11)
    assert round(b.cta_work_per_sm, 1) == 73.1 and round(w.cta_work_per_sm, 1) == 45.7
    assert ro.select_route({"buckets": b.total_us, "workqueue": w.total_us}, None, SEQ8, 4) == "workqueue"
    # and from the counters of the two routes themselves
    cb, _ = ro.bucket_route(SEQ8, 8, 4, 128, wq.Policy(tile_tokens=32, num_splits=32, route=wq.ROUTE_RECT), 1)
    cw = ro.single_route(SEQ8, 8, 4, 128, wq.Policy(tile_tokens=32, num_splits=20))
    assert ro.cost_of(cb, k).launch_us == b.launch_us and ro.cost_of(cb, k).merge_us == b.merge_us
    assert ro.cost_of(cw, k).launch_us == w.launch_us and ro.cost_of(cw, k).merge_us == w.merge_us


def test_p13_terms_closed_forms():
    k = ro.CostConstants(beta_gbps=1000.0, lambda_us=2.0, c_min=4.0, num_sms=10)
    # 1 GB/s = 1000 B/us: 5e6 B at 1000 GB/s = 5 us
    full = ro.route_cost(5_000_000, 0, 0, 40, k)                # C_r = 4 = C_min: factor exactly 1
    assert (full.stream_us, full.launch_us, full.merge_us, full.cta_work_per_sm) == (5.0, 0.0, 0.0, 4.0)
    assert ro.route_cost(5_000_000, 0, 0, 400, k).stream_us == 5.0            # above C_min: still 1
    half = ro.route_cost(5_000_000, 0, 0, 20, k)                # C_r = 2: factor C_min / C_r = 2
    assert half.stream_us == 10.0
    one = ro.route_cost(5_000_000, 1_000_000, 3, 1, k)          # one CTA on 10 SMs: factor 40
    assert one.stream_us == 200.0 and one.launch_us == 6.0 and one.merge_us == 1.0 and one.total_us == 207.0
    # linear in bytes and in launches, merge term independent of the occupancy factor
    a, b = ro.route_cost(3_000_000, 500_000, 2, 5, k), ro.route_cost(6_000_000, 1_000_000, 4, 5, k)
    assert b.total_us == pytest.approx(2 * a.total_us, rel=1e-15)


def test_p14_gates_and_margins():
    _, _, _, _, m8, m4, gate_tok, gate_g = _rows("cost_model_constants.txt")[0]
    assert (ro.MARGIN_B8, ro.MARGIN_B4, ro.GATE_MIN_TOKENS, ro.GATE_G) == (float(m8), float(m4), int(gate_tok), int(gate_g))
    long8, short8 = [20000] * 8, [16383] * 8
    assert ro.eligible(long8, 4) and not ro.eligible(short8, 4)
    assert ro.eligible([100, 16384], 4)                                     # the longest row decides (A25)
    assert not ro.eligible(long8, 1) and not ro.eligible(long8, 8)          # uncalibrated G
    est = {"base": 105.0, "workqueue": 100.0, "buckets": 101.0}
    assert ro.select_route(est, "base", long8, 4) == "workqueue"            # 1.05 clears the B8 margin
    assert ro.select_route({**est, "base": 104.9}, "base", long8, 4) == "base"
    assert ro.select_route(est, "base", short8, 4) == "base"                # 16K gate
    assert ro.select_route(est, "base", long8, 8) == "base"                 # G gate
    long4 = [20000] * 4
    assert ro.select_route({**est, "base": 149.0}, "base", long4, 4) == "base"        # B4: 1.50 needed
    assert ro.select_route({**est, "base": 150.0}, "base", long4, 4) == "workqueue"
    assert ro.select_route({**est, "base": 101.0}, "base", long4, 4, allow_b4=True) == "workqueue"   # the ablation flag
    assert ro.select_route(est, "base", [40000], 4) == "workqueue"          # B1 is a supported regime
    assert ro.select_route(est, None, short8, 8) == "workqueue"             # no baseline: the smallest estimate
    assert ro.select_route({"a": 1.0, "b": 1.0}, None, long8, 4) == "a"     # tie: first


def test_p15_makespan_form_reduces_to_the_papers_term_for_equal_tasks():
    """A27: with equal tasks and one task per CTA the makespan form IS the paper's stream term on
    both sides of C_r = C_min; with one oversized share it is that share at the lone-CTA rate."""
    k = ro.CostConstants(beta_gbps=1000.0, lambda_us=2.0, c_min=0.5, num_sms=100)
    # beta_cta = 1000 / (0.5 * 100) = 20 GB/s
    for tasks in (1, 10, 49, 50, 51, 100):
        kv = tasks * 2_000_000
        paper = ro.route_cost(kv, 0, 0, tasks, k).stream_us
        assert ro.stream_makespan_us(kv, 2_000_000, k) == pytest.approx(paper, rel=1e-12), tasks
    assert ro.stream_makespan_us(10_000_000, 4_000_000, k) == 200.0        # 4 MB at 20 GB/s beats 10 MB at 1000 GB/s
    assert ro.stream_makespan_us(100_000_000, 1_000_000, k) == 100.0
    # heads per CTA and the busiest share on a hand case: Hkv = 8, d = 128, 4 SMs
    assert [ro.heads_per_cta(8, rs, 148) for rs in (1, 15, 16, 31, 32, 62, 63, 125, 126, 148)] == [1, 1, 1, 1, 2, 2, 4, 4, 8, 8]
    assert ro.heads_per_cta(4, 1000, 148) == 4 and ro.heads_per_cta(32, 148, 148) == 8 and ro.heads_per_cta(2, 1, 148) == 1
    pol = wq.Policy(tile_tokens=32, num_splits=2)
    q = wq.build_workqueue([100, 1000], 8, pol)      # rows split in 2: 64+36 and 512+488 tokens; 4 pairs
    assert q.split_offsets[-1] == 4
    # 4 SMs: hg = 8 leaves 4 units = one wave; the largest unit is 512 tokens of 8 heads
    assert ro.max_share_bytes([100, 1000], 8, 128, q, 32, 4) == 512 * 2 * 8 * 128 * 2
    # 3 SMs: 4 units on 3 SMs = several waves: KV / SMs + the largest unit
    kv = 1100 * 4096
    assert ro.max_share_bytes([100, 1000], 8, 128, q, 32, 3) == kv // 3 + 512 * 4096
    # 5 SMs: 4 units of 8 heads cover only 80 % of them, so hg = 4: 8 units in 2 round-robin waves
    assert ro.heads_per_cta(8, 4, 5) == 4
    assert ro.max_share_bytes([100, 1000], 8, 128, q, 32, 5) == 2 * 512 * 2048
    # 148 SMs: nothing fills the machine, hg = 1: 32 units, one wave, 512 tokens of one head
    assert ro.max_share_bytes([100, 1000], 8, 128, q, 32, 148) == 512 * 512
