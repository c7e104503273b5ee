"""CPU-only checks of the C ABI: libpkv.so loads without a GPU, exports every symbol that
include/pkv.h declares, validates host-checkable arguments, and its HOST workqueue builder is
bit-exact against the pure-Python oracle.  No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2606_26666_b200 as pkv
from paper_2606_26666_b200 import binding
from oracle import workqueue_oracle as wq

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    text = open(os.path.join(ROOT, "include", "pkv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"PKV_API\s+[\w\s\*]+?\b(pkv_\w+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    syms = header_symbols()
    assert len(syms) >= 12
    lib = ctypes.CDLL(pkv.binding._build.LIB)
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(binding.EXPORTS) == syms


def test_version_and_struct_sizes():
    assert pkv.pkv_version() >> 16 == 2
    assert ctypes.sizeof(binding.pkv_task) == 20            # 5 x int32
    assert ctypes.sizeof(binding.pkv_split_policy) == 44
    assert ctypes.sizeof(binding.pkv_shape) == 80
    assert ctypes.sizeof(binding.pkv_counters) == 136


def shape(B, Hkv=8, Hq=32, max_pages=4096):
    return pkv.Shape(B=B, Hq=Hq, Hkv=Hkv, max_pages=max_pages, num_pages=1 << 20)


@pytest.mark.parametrize("bad,status", [
    (dict(d=96), pkv.PKV_ERR_UNSUPPORTED),
    (dict(page_size=48), pkv.PKV_ERR_UNSUPPORTED),
    (dict(Hq=48, Hkv=16), pkv.PKV_ERR_UNSUPPORTED),        # G = 3 not compiled in
    (dict(Hq=30, Hkv=8), pkv.PKV_ERR_INVALID_ARG),
    (dict(kv_strides=(4096, 4, 128)), pkv.PKV_ERR_INVALID_ARG),   # token stride not 16-byte multiple
])
def test_shape_validation(bad, status):
    kw = dict(B=2, Hq=32, Hkv=8, max_pages=8, num_pages=64)
    kw.update(bad)
    with pytest.raises(pkv.PkvError) as e:
        pkv.pkv_build_workqueue_host(pkv.Shape(**kw), pkv.Policy(num_splits=2), np.array([5, 6], np.int32))
    assert e.value.status == status
    assert pkv.pkv_last_error() != ""


@pytest.mark.parametrize("bad", [dict(tile_tokens=24), dict(tile_tokens=0), dict(num_splits=257),
                                 dict(split_mode=3), dict(split_mode=2, num_sms=0), dict(route=3), dict(merge_mode=2), dict(kernel=9),
                                 dict(split_mode=1, chunk_tiles=0), dict(num_splits=0, num_sms=0), dict(flags=1 << 20)])
def test_policy_validation(bad):
    with pytest.raises(pkv.PkvError) as e:
        pkv.pkv_build_workqueue_host(shape(1), pkv.Policy(**bad), np.array([100], np.int32))
    assert e.value.status == pkv.PKV_ERR_INVALID_ARG


def test_workspace_bytes_is_monotone_and_pure():
    a = pkv.pkv_workspace_bytes(shape(8), pkv.Policy(num_splits=4))
    b = pkv.pkv_workspace_bytes(shape(8), pkv.Policy(num_splits=16))
    assert 0 < a < b
    assert a == pkv.pkv_workspace_bytes(shape(8), pkv.Policy(num_splits=4))
    # partial states alone: slots * G * (d + 2) * 4 bytes (A11)
    assert b >= 8 * 8 * 16 * 4 * 130 * 4
    with pytest.raises(pkv.PkvError):
        pkv.pkv_workspace_bytes(shape(8), pkv.Policy(tile_tokens=17))


def oracle_tasks(seq_lens, Hkv, pol: pkv.Policy):
    opol = wq.Policy(tile_tokens=pol.tile_tokens, split_mode=pol.split_mode, num_splits=pol.num_splits,
                     chunk_tiles=pol.chunk_tiles, route=pol.route, merge_mode=pol.merge_mode, num_sms=pol.num_sms)
    q = wq.build_workqueue(list(map(int, seq_lens)), Hkv, opol)
    return np.array(q.tasks, dtype=np.int32).reshape(-1, 5), np.array(q.split_offsets, dtype=np.int32), q


POLICIES = [
    pkv.Policy(tile_tokens=32, num_splits=1),
    pkv.Policy(tile_tokens=32, num_splits=20),
    pkv.Policy(tile_tokens=64, num_splits=7),
    pkv.Policy(tile_tokens=16, num_splits=256),
    pkv.Policy(tile_tokens=32, num_splits=0, num_sms=28),
    pkv.Policy(tile_tokens=32, num_splits=0, num_sms=148),
    pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=16),
    pkv.Policy(tile_tokens=128, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=12, chunk_tiles=3),
    pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=148),
    pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=148),
    pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=28),
    pkv.Policy(tile_tokens=64, split_mode=pkv.SPLIT_BALANCED, num_splits=5, num_sms=7),
    pkv.Policy(tile_tokens=32, num_splits=20, route=pkv.ROUTE_RECT),
    pkv.Policy(tile_tokens=64, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=9, chunk_tiles=4, route=pkv.ROUTE_RECT),
]


@pytest.mark.parametrize("pol", POLICIES, ids=lambda p: "T%d_m%d_S%d_c%d_r%d_sm%d" % (
    p.tile_tokens, p.split_mode, p.num_splits, p.chunk_tiles, p.route, p.num_sms))
def test_host_builder_bit_exact_vs_python_oracle(pol):
    rng = np.random.Generator(np.random.PCG64(1234))
    cases = [[0], [1], [0, 0, 0], [31, 32, 33, 0, 1], [65536], list(rng.integers(0, 70000, size=8)),
             list(rng.integers(0, 3000, size=37)), [16384 + i for i in range(8)], []]
    for Hkv in (8, 4):
        for lens in cases:
            lens = np.array(lens, dtype=np.int32)
            ref_t, ref_o, _ = oracle_tasks(lens, Hkv, pol)
            got_t, got_o = pkv.pkv_build_workqueue_host(shape(len(lens), Hkv=Hkv), pol, lens)
            assert got_t.shape == ref_t.shape, (lens, Hkv)
            assert np.array_equal(got_t, ref_t), (lens, Hkv)
            assert np.array_equal(got_o, ref_o), (lens, Hkv)


def test_host_builder_on_the_trace_configs():
    import pkv_inputs
    for w in (pkv_inputs.config3(), pkv_inputs.config4(), pkv_inputs.config4_b4(), pkv_inputs.config5()):
        for step in (0, w.steps):
            lens = w.seq_lens_at(step)
            for pol in (pkv.Policy(tile_tokens=32, num_splits=20),
                        pkv.Policy(tile_tokens=64, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=8),
                        pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=148),
                        pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=148)):
                ref_t, ref_o, _ = oracle_tasks(lens, w.Hkv, pol)
                got_t, got_o = pkv.pkv_build_workqueue_host(shape(w.B, Hkv=w.Hkv), pol, lens)
                assert np.array_equal(got_t, ref_t) and np.array_equal(got_o, ref_o), (w.name, step)


def test_tasks_cap_too_small_reports_needed_count():
    s, pol = shape(1), pkv.Policy(num_splits=4)
    lens = np.array([1000], np.int32)
    tasks = np.zeros((3, 5), np.int32)
    off = np.zeros(2, np.int32)
    n = ctypes.c_int32(0)
    st = binding._lib.pkv_build_workqueue_host(ctypes.byref(s.c()), ctypes.byref(pol.c()), lens.ctypes.data,
                                               tasks.ctypes.data, 3, off.ctypes.data, ctypes.byref(n))
    assert st == pkv.PKV_ERR_WORKSPACE and n.value == 32


def test_bucket_plan_and_counters_match_the_route_oracle():
    """pkv_plan_buckets_host / pkv_bucket_counters_host against oracle/route_oracle.py (PAPER.md:71,
    93, 204-206; readings A22, A23): grouping, order, and Table 4's bucket row (16.00 launches,
    8.00 merge launches, 2048 tasks, 4.06 MB)."""
    from oracle import route_oracle as ro
    rng = np.random.Generator(np.random.PCG64(5))
    cases = [[5000, 0, 4999, 5000, 17, 4990, 32], [0, 0], [7], list(rng.integers(0, 70000, size=64)),
             [8192, 16384, 32768, 65536] * 3, [32768] * 8]
    for lens in cases:
        for gran in (1, 16, 1024, 8192, 1 << 20):
            index, offs, blen = pkv.pkv_plan_buckets_host(np.array(lens, np.int32), gran)
            want = ro.group_buckets(lens, gran)
            assert len(offs) == len(want) + 1 and list(blen) == [k for k, _ in want]
            assert [list(index[offs[b]:offs[b + 1]]) for b in range(len(want))] == [rows for _, rows in want]
            assert sorted(index) == list(range(len(lens)))
            assert list(index[offs[-1]:]) == [i for i, n in enumerate(lens) if n <= 0]
            for pol in (pkv.Policy(tile_tokens=32, num_splits=32, route=pkv.ROUTE_RECT),
                        pkv.Policy(tile_tokens=32, num_splits=5, route=pkv.ROUTE_WORKQUEUE, merge_mode=pkv.MERGE_FUSED),
                        pkv.Policy(tile_tokens=16, num_splits=1, route=pkv.ROUTE_RECT)):
                c = pkv.pkv_bucket_counters_host(shape(len(lens)), pol, np.array(lens, np.int32), gran)
                w, _ = ro.bucket_route(lens, 8, 4, 128, wq.Policy(tile_tokens=pol.tile_tokens, num_splits=pol.num_splits,
                                                                   route=pol.route, merge_mode=pol.merge_mode), gran)
                assert (c["decode_launches"] + c["merge_launches"], c["merge_launches"], c["tasks"], c["empty_tasks"],
                        c["merge_bytes"], c["useful_kv_bytes"]) == (w.launches, w.merge_launches, w.tasks, w.empty_tasks,
                                                                    w.merge_bytes, w.useful_kv_bytes), (lens, gran, pol)
    seq = [16384 + 977 * i for i in range(8)]
    c = pkv.pkv_bucket_counters_host(shape(8), pkv.Policy(tile_tokens=32, num_splits=32, route=pkv.ROUTE_RECT),
                                     np.array(seq, np.int32), 1)
    assert (c["decode_launches"] + c["merge_launches"], c["merge_launches"], c["tasks"]) == (16, 8, 2048)
    assert "%.2f" % (c["merge_bytes"] / 2 ** 20) == "4.06"


def test_cost_model_matches_the_route_oracle():
    """pkv_estimate_cost against oracle/route_oracle.py: every term of T_r, C_r, and
    the makespan form (A27), for single launch pairs and for the bucket route, with the paper's
    constants and with the B200 defaults; Table 4's 16-vs-2 launch case prefers the workqueue."""
    from oracle import route_oracle as ro
    rng = np.random.Generator(np.random.PCG64(9))
    models = [pkv.CostModel(331.2, 8.19, 4.0, 28), pkv.pkv_default_cost_model(148)]
    assert (models[1].beta_gbps, models[1].num_sms) == (7060.0, 148)
    cases = [[16384 + 977 * i for i in range(8)], [32768], [700, 0, 33, 20000, 5, 64000], list(rng.integers(0, 70000, size=40)), [0, 0]]
    pols = [pkv.Policy(tile_tokens=32, num_splits=20), pkv.Policy(tile_tokens=32, num_splits=32, route=pkv.ROUTE_RECT),
            pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0),
            pkv.Policy(tile_tokens=32, num_splits=1), pkv.Policy(tile_tokens=32, num_splits=6, merge_mode=pkv.MERGE_FUSED)]
    for m in models:
        k = ro.CostConstants(m.beta_gbps, m.lambda_us, m.c_min, m.num_sms)
        for lens in cases:
            sh = shape(len(lens))
            for pol in pols:
                opol = wq.Policy(tile_tokens=pol.tile_tokens, split_mode=pol.split_mode, num_splits=pol.num_splits,
                                 route=pol.route, merge_mode=pol.merge_mode, num_sms=m.num_sms)
                e = pkv.pkv_estimate_cost(sh, pol, np.array(lens, np.int32), 0, m)
                c = ro.single_route(lens, 8, 4, 128, opol)
                t = ro.cost_of(c, k)
                q = wq.build_workqueue(lens, 8, opol)
                share = ro.max_share_bytes(lens, 8, 128, q, pol.tile_tokens, m.num_sms)
                assert (e["kv_bytes"], e["merge_bytes"], e["tasks"], e["launches"], e["max_share_bytes"]) == (
                    c.useful_kv_bytes, c.merge_bytes, c.tasks, c.launches, share), (lens, pol)
                for got, want in ((e["stream_us"], t.stream_us), (e["launch_us"], t.launch_us), (e["merge_us"], t.merge_us),
                                  (e["total_us"], t.total_us), (e["cta_work_per_sm"], t.cta_work_per_sm),
                                  (e["makespan_us"], ro.stream_makespan_us(c.useful_kv_bytes, share, k,
                                                                            ro.heads_per_cta(8, q.split_offsets[-1], m.num_sms) if q.split_offsets[-1] else 8))):
                    assert got == pytest.approx(want, rel=1e-12, abs=1e-300), (lens, pol)
                if pol.split_mode == pkv.SPLIT_BALANCED:
                    continue
                for gran in (1, 4096):
                    e = pkv.pkv_estimate_cost(sh, pol, np.array(lens, np.int32), gran, m)
                    cb, _ = ro.bucket_route(lens, 8, 4, 128, opol, gran)
                    tb = ro.cost_of(cb, k)
                    assert (e["tasks"], e["launches"], e["merge_bytes"]) == (cb.tasks, cb.launches, cb.merge_bytes)
                    assert e["total_us"] == pytest.approx(tb.total_us, rel=1e-12, abs=1e-300)
    # Table 4 with the paper's constants: exact buckets at split 32 vs the workqueue at split 20
    seq = np.array([16384 + 977 * i for i in range(8)], np.int32)
    b = pkv.pkv_estimate_cost(shape(8), pols[1], seq, 1, models[0])
    w = pkv.pkv_estimate_cost(shape(8), pols[0], seq, 0, models[0])
    assert b["launches"] == 16 and w["launches"] == 2 and w["total_us"] < b["total_us"]
    assert b["launch_us"] - w["launch_us"] == pytest.approx(14 * 8.19, rel=1e-12)


def test_choose_policy_picks_the_smallest_estimate():
    """pkv_choose_policy = argmin of makespan_total_us over {BALANCED, FIXED_COUNT S = 1..128}
    (first wins ties), restated here with pkv_estimate_cost; and the choices that matter on B200:
    one long row is never left unsplit, a large uniform batch is, a ragged batch gets BALANCED."""
    m = pkv.pkv_default_cost_model(148)
    base = pkv.Policy(split_mode=pkv.SPLIT_AUTO, num_splits=0, tile_tokens=16)
    rng = np.random.Generator(np.random.PCG64(11))
    for lens in ([32768], [300], list(rng.integers(1024, 65536, size=128)), [700, 22000, 31000, 450, 900, 17000, 260, 30000],
                 [100] * 8, [0, 0, 5]):
        sh = shape(len(lens))
        got, est = pkv.pkv_choose_policy(sh, np.array(lens, np.int32), m, base)
        cands = [pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0)] + \
                [pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_COUNT, num_splits=1 << c) for c in range(8)]
        s_fit = min(256, 148 // len(lens))          # Hkv = 8 in one head group
        if s_fit >= 2 and s_fit & (s_fit - 1):
            cands.append(pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_COUNT, num_splits=s_fit))
        ests = [pkv.pkv_estimate_cost(sh, p, np.array(lens, np.int32), 0, m) for p in cands]
        costs = [e["makespan_total_us"] for e in ests]
        # within 1 % of the smallest estimate: the fullest machine, then the smaller estimate, then the first
        near = [i for i in range(len(cands)) if costs[i] <= 1.01 * min(costs)]
        pick = max(near, key=lambda i: (min(ests[i]["units"], 148), -costs[i], cands[i].split_mode == pkv.SPLIT_FIXED_COUNT, -i))
        best = cands[pick]
        assert (got.split_mode, got.num_splits, got.tile_tokens) == (best.split_mode, best.num_splits, best.tile_tokens), lens
        assert est["makespan_total_us"] == costs[pick]
    one, _ = pkv.pkv_choose_policy(shape(1), np.array([32768], np.int32), m, base)
    assert one.split_mode == pkv.SPLIT_BALANCED or one.num_splits >= 16
    big, _ = pkv.pkv_choose_policy(shape(8), np.array([100] * 8, np.int32), m, base)
    assert big.split_mode == pkv.SPLIT_FIXED_COUNT and big.num_splits == 1
