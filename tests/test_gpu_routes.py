"""GPU tests of the length-bucket route and indexed rows (DESIGN.md
readings A22, A23): pkv_decode_indexed decodes a subset of the batch's rows in place, and
pkv_decode_buckets issues one launch pair per route length.  Outputs against the FP64 oracle,
queues and launch counts against the workqueue / route oracles."""
import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
import pkv_inputs
from gpu_helpers import DevProblem, oracle_attention, oracle_policy, to_dev
from helpers import assert_within_tolerance, make_problem
from oracle import route_oracle as ro
from oracle import workqueue_oracle as wq

pytestmark = pytest.mark.gpu

LENS = [700, 33, 0, 2000, 16, 257, 700, 1, 4097, 700, 33, 31]


@pytest.mark.parametrize("kernel", [pkv.KERNEL_TMA_MMA, pkv.KERNEL_SIMT])
@pytest.mark.parametrize("fused_build", [True, False])
def test_indexed_rows_decode_a_subset_in_place(kernel, fused_build):
    """Rows outside the index keep whatever out / lse held; indexed rows (in any order, with an
    empty row among them) match the oracle; the queue in the workspace is the oracle's queue of the
    indexed rows' lengths, in launch-row order."""
    p = make_problem(LENS, seed=81)
    dp = DevProblem(p)
    ref, ref_lse = oracle_attention(p)
    for index in ([3], [8, 0, 2, 5], [11, 10, 9, 8, 7, 6, 5, 4, 3, 2, 1, 0], [1, 4, 7, 2]):
        for pol in (pkv.Policy(tile_tokens=32, num_splits=4, kernel=kernel),
                    pkv.Policy(tile_tokens=32, num_splits=3, kernel=kernel, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT),
                    pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=12, kernel=kernel)):
            pol.flags = 0 if fused_build else pkv.FLAG_SEPARATE_BUILD
            sub = pkv.Shape(B=len(index), Hq=p.Hq, Hkv=p.Hkv, max_pages=dp.shape.max_pages, num_pages=dp.shape.num_pages)
            ws = pkv.alloc_workspace(dp.shape, pol)
            dp.out.fill_(7.0)
            dp.lse.fill_(7.0)
            pkv.pkv_decode_indexed(sub, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, to_dev(np.array(index, np.int32)), dp.out, dp.lse,
                                   scale=p.scale, workspace=ws)
            torch.cuda.synchronize()
            out, lse = dp.out.cpu().numpy().astype(np.float64), dp.lse.cpu().numpy().astype(np.float64)
            rest = [i for i in range(p.B) if i not in index]
            assert np.all(out[rest] == 7.0) and np.all(lse[rest] == 7.0), (index, pol)
            assert_within_tolerance(out[index], ref[index], "index %s %s" % (index, pol))
            fin = np.isfinite(ref_lse[index])
            assert np.abs(lse[index][fin] - ref_lse[index][fin]).max(initial=0.0) <= 2e-3
            assert np.array_equal(np.isneginf(lse[index]), np.isneginf(ref_lse[index]))
            tasks, offs = pkv.pkv_read_workqueue(sub, pol, ws)
            want = wq.build_workqueue([LENS[i] for i in index], p.Hkv, oracle_policy(pol))
            assert tasks.tolist() == [list(t) for t in want.tasks] and offs.tolist() == want.split_offsets


@pytest.mark.parametrize("gran", [1, 16, 1024, 1 << 20])
def test_bucket_route_matches_the_oracle_and_the_workqueue_route(gran):
    """One launch pair per route length (A23): every row's output within tolerance of the oracle
    (rows of no bucket: zeros), launches as oracle/route_oracle.py counts them."""
    p = make_problem(LENS, seed=83)
    dp = DevProblem(p)
    ref, ref_lse = oracle_attention(p)
    lens = np.array(LENS, np.int32)
    index, offs, blen = pkv.pkv_plan_buckets_host(lens, gran)
    for pol in (pkv.Policy(tile_tokens=32, num_splits=4, route=pkv.ROUTE_RECT),
                pkv.Policy(tile_tokens=32, num_splits=6, route=pkv.ROUTE_WORKQUEUE, merge_mode=pkv.MERGE_FUSED)):
        ws = pkv.alloc_workspace(dp.shape, pol)
        dp.out.fill_(float("nan"))
        dp.lse.fill_(float("nan"))
        pkv.pkv_decode_buckets(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, to_dev(index), offs, dp.out, dp.lse,
                               scale=p.scale, workspace=ws)
        torch.cuda.synchronize()
        out, lse = dp.out.cpu().numpy().astype(np.float64), dp.lse.cpu().numpy().astype(np.float64)
        assert not np.isnan(out).any() and not np.isnan(lse).any()
        assert_within_tolerance(out, ref, "gran %d %s" % (gran, pol))
        assert np.array_equal(np.isneginf(lse), np.isneginf(ref_lse))
        c = pkv.pkv_bucket_counters_host(dp.shape, pol, lens, gran)
        w, _ = ro.bucket_route(LENS, p.Hkv, p.Hq // p.Hkv, p.d, oracle_policy(pol), gran)
        assert c["decode_launches"] + c["merge_launches"] == w.launches and c["tasks"] == w.tasks


def test_table4_launch_fan_out_on_a_bimodal_b8_step():
    """Table 4 in kind: a B = 8 step whose rows all have distinct lengths costs
    8 + 8 launches on exact length buckets at split 32 and 1 + 1 on the compact workqueue at split 20;
    both routes give the oracle's result."""
    w = pkv_inputs.trace("bimodal", seed=pkv_inputs.REPORT_SEEDS[0], B=8, steps=0)
    lens = (w.seq_lens // 8).astype(np.int32)          # same shape of trace at an eighth of the length
    assert len(set(lens.tolist())) == 8
    p = make_problem(list(lens), seed=85)
    dp = DevProblem(p)
    ref, _ = oracle_attention(p)
    pb = pkv.Policy(tile_tokens=32, num_splits=32, route=pkv.ROUTE_RECT)
    pw = pkv.Policy(tile_tokens=32, num_splits=20, route=pkv.ROUTE_WORKQUEUE)
    index, offs, _ = pkv.pkv_plan_buckets_host(lens, 1)
    assert len(offs) - 1 == 8
    cb = pkv.pkv_bucket_counters_host(dp.shape, pb, lens, 1)
    assert (cb["decode_launches"] + cb["merge_launches"], cb["merge_launches"]) == (16, 8)
    ws = pkv.alloc_workspace(dp.shape, pb)
    pkv.pkv_decode_buckets(dp.shape, pb, dp.q, dp.k, dp.v, dp.bt, dp.sl, to_dev(index), offs, dp.out, None, scale=p.scale, workspace=ws)
    torch.cuda.synchronize()
    assert_within_tolerance(dp.out.cpu().numpy().astype(np.float64), ref, "buckets")
    out, _, ws = dp.decode(pw)
    assert_within_tolerance(out, ref, "workqueue")
    cw = pkv.pkv_get_counters(dp.shape, pw, ws)
    assert (cw["decode_launches"] + cw["merge_launches"], cw["merge_launches"]) == (2, 1)
    assert (cw["launched_decode"], cw["launched_merge"]) == (1, 1)


@pytest.mark.parametrize("family", ["bimodal", "bucketed"])
def test_serving_loop_with_arrivals_and_finishes(family):
    """A continuous-decode loop: requests arrive, grow by one token per step and finish;
    slots go empty and are re-used with other pages.  Every step runs through pkv.HostDecoder with
    PKV_SPLIT_AUTO (the cost model re-plans per step) on one (staging, scratch) pair; every third step
    is checked against the oracle, and all rows of empty slots must be zero."""
    from gpu_helpers import oracle_attention
    from helpers import Problem, default_scale
    tr = pkv_inputs.ServingTrace(family, seed=21, requests=14, max_active=6, decode_lo=4, decode_hi=12, prompt_div=8)
    k = pkv_inputs.fill_normal_f16((tr.num_pages, 16, 8, 128), 31)
    v = pkv_inputs.fill_normal_f16((tr.num_pages, 16, 8, 128), 32)
    q = pkv_inputs.fill_normal_f16((6, 32, 128), 33)
    dk, dv = to_dev(k), to_dev(v)
    shape = pkv.Shape(B=6, Hq=32, Hkv=8, max_pages=tr.max_pages, num_pages=tr.num_pages)
    pol = pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_AUTO, num_splits=0)
    nb = pkv.pkv_host_scratch_bytes(shape, pol)
    staging = torch.zeros(nb, dtype=torch.uint8).pin_memory()
    scratch = torch.empty(nb, dtype=torch.uint8, device="cuda")
    ws = pkv.alloc_workspace(shape, pol)
    out = torch.full((6, 32, 128), float("nan"), dtype=torch.float16).pin_memory()
    dec = pkv.HostDecoder(shape, pol, dk, dv, staging, scratch, ws, default_scale(128))
    steps = empties = checked = 0
    for st in tr.steps():
        lens = np.ascontiguousarray(st.seq_lens)
        table = np.ascontiguousarray(st.block_table)
        dec(q.ctypes.data, table.ctypes.data, lens.ctypes.data, out.data_ptr())
        got = out.numpy().astype(np.float64)
        assert not np.isnan(got).any()
        for s in range(6):
            if lens[s] == 0:
                assert np.all(got[s] == 0)
                empties += 1
        if st.step % 3 == 0 or st.started or st.finished:
            p = Problem(q=q, k_cache=k, v_cache=v, block_table=table, seq_lens=lens, Hkv=8, page_size=16, scale=default_scale(128))
            assert_within_tolerance(got, oracle_attention(p)[0], "step %d" % st.step)
            checked += 1
        steps += 1
    assert steps > 20 and empties > 0 and checked > 10
