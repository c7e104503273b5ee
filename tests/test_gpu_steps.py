"""GPU tests of whole decode STEPS as a serving loop issues them: many consecutive steps in one
CUDA graph with programmatic dependent launch on and no host synchronisation in between
(the overlapped replay bench.py times), the device-side validation of
device-resident inputs (every bound derives from N_i), the launch marks behind
pkv_counters.launched_*, and a second device in the same process."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
from gpu_helpers import DevProblem, oracle_attention, oracle_policy, to_dev
from helpers import assert_within_tolerance, make_problem
from oracle import workqueue_oracle as wq
from pkv_inputs import PAD_PAGE

pytestmark = pytest.mark.gpu


def _multi_step_graph(dp, p, pol, lens0, steps, pdl):
    """Captures `steps` consecutive pkv_decode calls in ONE graph: step t reads row t of a device
    table of lengths (N_i + t) and writes row t of [steps, B, Hq, d] / [steps, B, Hq] outputs.
    One replay, no host sync between the steps.  Returns (out, lse) as float64 numpy arrays."""
    B = len(lens0)
    lens_all = np.stack([lens0 + t for t in range(steps)]).astype(np.int32)
    sl_all = to_dev(lens_all)
    out = torch.full((steps, B, p.Hq, p.d), float("nan"), dtype=torch.float16, device="cuda")
    lse = torch.full((steps, B, p.Hq), float("nan"), dtype=torch.float32, device="cuda")
    pol = dataclasses.replace(pol, flags=pol.flags | (0 if pdl else pkv.FLAG_NO_PDL))
    ws = pkv.alloc_workspace(dp.shape, pol)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        pkv.pkv_decode(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, sl_all[0], out[0], lse[0], scale=p.scale,
                       workspace=ws, stream=s)      # warm-up outside capture (function attributes)
        s.synchronize()
        out.fill_(float("nan"))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for t in range(steps):
                pkv.pkv_decode(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, sl_all[t], out[t], lse[t],
                               scale=p.scale, workspace=ws, stream=torch.cuda.current_stream())
        g.replay()
        g.replay()      # twice: self-resetting counters, workspace reused across replays
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("mm", [pkv.MERGE_SEPARATE, pkv.MERGE_FUSED])
@pytest.mark.parametrize("mode", [pkv.SPLIT_FIXED_COUNT, pkv.SPLIT_BALANCED])
def test_overlapped_multi_step_graph_every_step_checked(mm, mode):
    """12 consecutive steps in one graph, PDL on: the merge of step t overlaps the start of step
    t+1 (race-tolerant early reads of seq_lens / split_offsets, re-validated after the dependency
    wait).  Every step's output is compared with the oracle, and bitwise with the same graph
    launched without programmatic dependent launch."""
    steps = 12
    lens0 = np.array([60, 1000, 31, 257, 0, 4090, 15, 2047], dtype=np.int32)   # tile/page crossings inside 12 steps
    p = make_problem(lens0, seed=195, reserve_extra=steps)
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=16 if mode == pkv.SPLIT_BALANCED else 32, split_mode=mode,
                     num_splits=0 if mode == pkv.SPLIT_BALANCED else 5, merge_mode=mm,
                     num_sms=24 if mode == pkv.SPLIT_BALANCED else 0)
    o_on, l_on = _multi_step_graph(dp, p, pol, lens0, steps, True)
    o_off, l_off = _multi_step_graph(dp, p, pol, lens0, steps, False)
    assert np.array_equal(o_on, o_off) and np.array_equal(l_on, l_off)
    for t in range(steps):
        p.seq_lens = (lens0 + t).astype(np.int32)
        ref, ref_lse = oracle_attention(p)
        assert_within_tolerance(o_on[t], ref, "step %d" % t)
        fin = np.isfinite(ref_lse)
        assert np.abs(l_on[t][fin] - ref_lse[fin]).max() <= 2e-3


def test_validate_flag_reports_bad_lengths_and_page_ids():
    """PKV_FLAG_VALIDATE: a length the block table cannot describe and a
    page id outside the pool are recorded in pkv_counters.error_word, the kernels stay inside the
    caller's buffers, and the rows without a fault are still right."""
    lens = np.array([300, 77, 1000], dtype=np.int32)
    for kernel in (pkv.KERNEL_TMA_MMA, pkv.KERNEL_SIMT):
        for fused_build in (True, False):
            p = make_problem(lens, seed=61)
            ref = oracle_attention(p)[0]
            max_tokens = p.block_table.shape[1] * 16
            pol = pkv.Policy(tile_tokens=32, num_splits=3, kernel=kernel,
                             flags=pkv.FLAG_VALIDATE | (0 if fused_build else pkv.FLAG_SEPARATE_BUILD))
            if True:
                # clean inputs: no error bit
                dp = DevProblem(p)
                out, _, ws = dp.decode(pol)
                assert pkv.pkv_get_counters(dp.shape, pol, ws)["error_word"] == 0
                assert_within_tolerance(out, ref)
                # row 1 claims more tokens than its table row holds
                bad = lens.copy()
                bad[1] = max_tokens + 1234
                dp.sl.copy_(to_dev(bad))
                out, _, ws = dp.decode(pol)
                # the row is decoded as if it had max_tokens tokens, so its padding entries are
                # dereferenced too (and replaced by page 0): both bits
                assert pkv.pkv_get_counters(dp.shape, pol, ws)["error_word"] == pkv.DEVERR_SEQ_LEN | pkv.DEVERR_PAGE_ID
                assert_within_tolerance(out[[0, 2]], ref[[0, 2]])
                # the same with a table row that is valid end to end: the length fault alone
                bt = p.block_table.copy()
                bt[1, :] = bt[1, 0]
                dp.bt.copy_(to_dev(bt))
                out, _, ws = dp.decode(pol)
                assert pkv.pkv_get_counters(dp.shape, pol, ws)["error_word"] == pkv.DEVERR_SEQ_LEN
                assert_within_tolerance(out[[0, 2]], ref[[0, 2]])
                # row 2 points at a page outside the pool (row 1 keeps its padding entries unread)
                dp.sl.copy_(to_dev(lens))
                bt = p.block_table.copy()
                bt[2, 5] = p.k_cache.shape[0] + 7
                dp.bt.copy_(to_dev(bt))
                out, _, ws = dp.decode(pol)
                assert pkv.pkv_get_counters(dp.shape, pol, ws)["error_word"] == pkv.DEVERR_PAGE_ID
                assert_within_tolerance(out[[0, 1]], ref[[0, 1]])
                assert np.all(p.block_table[1, -(-77 // 16):] == PAD_PAGE)      # padding never dereferenced
                # sticky until the workspace is initialised again: a clean step on the same workspace
                dp.bt.copy_(to_dev(p.block_table))
                out, _, _ = dp.decode(pol, ws=ws)
                assert pkv.pkv_get_counters(dp.shape, pol, ws)["error_word"] == pkv.DEVERR_PAGE_ID
                assert_within_tolerance(out, ref)


def test_launch_marks_count_what_was_really_launched():
    """pkv_counters.launched_*: each kernel leaves its mark.  On the device path the merge kernel is
    launched whenever the policy allows several splits per row -- even if no row has more than one
    -- and the decode kernel even when every row is empty; the scheduler-derived counters
    (Table 4 definitions) say 0 there."""
    p = make_problem([20, 0, 31], seed=63)          # one tile per row: n_i <= 1
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=32, num_splits=4)
    _, _, ws = dp.decode(pol)
    c = pkv.pkv_get_counters(dp.shape, pol, ws)
    assert (c["decode_launches"], c["merge_launches"]) == (1, 0)
    assert (c["launched_build"], c["launched_decode"], c["launched_merge"]) == (0, 1, 1)
    pol_sb = dataclasses.replace(pol, flags=pkv.FLAG_SEPARATE_BUILD)
    _, _, ws = dp.decode(pol_sb)
    c = pkv.pkv_get_counters(dp.shape, pol_sb, ws)
    assert (c["launched_build"], c["launched_decode"], c["launched_merge"]) == (1, 1, 1)
    pol1 = pkv.Policy(tile_tokens=32, num_splits=1)
    _, _, ws = dp.decode(pol1)
    c = pkv.pkv_get_counters(dp.shape, pol1, ws)
    assert (c["launched_build"], c["launched_decode"], c["launched_merge"]) == (0, 1, 0)
    pf = pkv.Policy(tile_tokens=32, num_splits=4, merge_mode=pkv.MERGE_FUSED, kernel=pkv.KERNEL_SIMT)
    _, _, ws = dp.decode(pf)
    c = pkv.pkv_get_counters(dp.shape, pf, ws)
    assert (c["launched_build"], c["launched_decode"], c["launched_merge"]) == (1, 1, 0)
    p0 = make_problem([0, 0], seed=64)
    dp0 = DevProblem(p0)
    out, _, ws = dp0.decode(pol)
    c = pkv.pkv_get_counters(dp0.shape, pol, ws)
    assert c["decode_launches"] == 0 and c["launched_decode"] == 1 and np.all(out == 0)


def test_second_device_in_the_same_process():
    """The TMA kernel's dynamic shared-memory opt-in is a per-device attribute: after a launch on
    device 0, device 1 must still get its own opt-in."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one device")
    p = make_problem([700, 33, 2000], seed=65)
    ref = oracle_attention(p)[0]
    pol = pkv.Policy(tile_tokens=32, num_splits=4)
    for dev in (0, 1, 0):
        with torch.cuda.device(dev):
            q, k, v = (torch.from_numpy(a).cuda() for a in (p.q, p.k_cache, p.v_cache))
            bt, sl = torch.from_numpy(p.block_table).cuda(), torch.from_numpy(p.seq_lens).cuda()
            shape = pkv.Shape(B=p.B, Hq=p.Hq, Hkv=p.Hkv, max_pages=p.block_table.shape[1], num_pages=p.k_cache.shape[0])
            out = torch.zeros((p.B, p.Hq, p.d), dtype=torch.float16, device="cuda")
            ws = pkv.alloc_workspace(shape, pol, device="cuda:%d" % dev)
            pkv.pkv_decode(shape, pol, q, k, v, bt, sl, out, None, scale=p.scale, workspace=ws)
            torch.cuda.synchronize()
            assert_within_tolerance(out.cpu().numpy().astype(np.float64), ref, "device %d" % dev)


@pytest.mark.parametrize("mode", [pkv.SPLIT_FIXED_COUNT, pkv.SPLIT_BALANCED])
def test_block_table_and_lengths_rewritten_right_before_every_step(mode):
    """The kernel right before pkv_decode rewrites the block table AND the lengths in every step of
    one graph (PDL on).  Before its dependency wait the decode kernel looks at both with
    race-tolerant loads -- for the speculative plan and for the L2 prefetch of its first pages
     -- so what it sees there is the PREVIOUS step's table; every value the
    result depends on must be loaded after the wait.  Two page assignments of the same logical
    content alternate (pool = [pages | pages rolled by one]); every step is checked against the
    oracle and bitwise against the same graph without programmatic launch and without prefetch."""
    steps = 10
    lens0 = np.array([3000, 40, 1111, 0, 257, 4090], dtype=np.int32)
    p = make_problem(list(lens0 + steps), seed=71)
    n = p.k_cache.shape[0]
    p.k_cache = np.concatenate([p.k_cache, np.roll(p.k_cache, 1, axis=0)])
    p.v_cache = np.concatenate([p.v_cache, np.roll(p.v_cache, 1, axis=0)])
    tab_a = p.block_table.copy()
    tab_b = np.where(tab_a == PAD_PAGE, PAD_PAGE, n + (tab_a.astype(np.int64) + 1) % n).astype(np.int32)
    dp = DevProblem(p)
    tabs = to_dev(np.stack([tab_a, tab_b]))
    lens_all = to_dev(np.stack([lens0 + t for t in range(steps)]).astype(np.int32))
    base = pkv.Policy(tile_tokens=16 if mode == pkv.SPLIT_BALANCED else 32, split_mode=mode,
                      num_splits=0 if mode == pkv.SPLIT_BALANCED else 6, num_sms=40 if mode == pkv.SPLIT_BALANCED else 0)
    results = []
    for pol in (base, dataclasses.replace(base, flags=pkv.FLAG_NO_PDL, prefetch_kb=-1)):
        out = torch.full((steps, p.B, p.Hq, p.d), float("nan"), dtype=torch.float16, device="cuda")
        ws = pkv.alloc_workspace(dp.shape, pol)
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            pkv.pkv_decode(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, out[0], None, scale=p.scale, workspace=ws, stream=s)
            s.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                for t in range(steps):
                    dp.bt.copy_(tabs[t % 2])          # the predecessor kernels of step t
                    dp.sl.copy_(lens_all[t])
                    pkv.pkv_decode(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, out[t], None, scale=p.scale,
                                   workspace=ws, stream=torch.cuda.current_stream())
            g.replay()
            g.replay()
        torch.cuda.synchronize()
        results.append(out.cpu().numpy().astype(np.float64))
    assert np.array_equal(results[0], results[1])
    p.block_table = tab_a
    for t in range(steps):
        p.seq_lens = (lens0 + t).astype(np.int32)
        assert_within_tolerance(results[0][t], oracle_attention(p)[0], "step %d" % t)
