"""GPU parity: the CUDA path (through the C ABI) against the FP64 oracle, element by element,
on the same seeded inputs.  Tolerance = BASELINE.json north_star with DESIGN.md reading A15:
max abs <= 2e-3, floored max rel <= 1e-2, mean abs <= 3e-4.  Integer work
(tasks, split_offsets, counters, token counts) is compared bit-exactly."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
import pkv_inputs
from gpu_helpers import DevProblem, oracle_attention, oracle_policy, read_partials, sm_count, to_dev
from helpers import (assert_within_tolerance, default_scale, make_problem, permute_pool, token_location, Problem)
from oracle import pkv_oracle, workqueue_oracle as wq
from pkv_inputs import PAD_PAGE

pytestmark = pytest.mark.gpu

KERNELS = [pkv.KERNEL_TMA_MMA, pkv.KERNEL_SIMT]
RAGGED = [1, 2, 15, 16, 17, 31, 32, 33, 100, 0, 257, 700]


def check(dp, pol, ref=None, what=""):
    out, lse, ws = dp.decode(pol)
    if ref is None:
        ref = oracle_attention(dp.p)
    assert not np.isnan(out).any(), what
    m = assert_within_tolerance(out, ref[0], what)
    fin = np.isfinite(ref[1])
    assert np.array_equal(np.isneginf(lse), np.isneginf(ref[1])), what
    assert np.abs(lse[fin] - ref[1][fin]).max(initial=0.0) <= 2e-3, what
    return out, lse, ws, m


@pytest.mark.parametrize("kernel", KERNELS)
def test_config1(kernel):
    """BASELINE.json configs[0]: B=1, N=256, 16 pages of a 64-page pool, no splitting."""
    w = pkv_inputs.config1()
    p = Problem(q=pkv_inputs.fill_normal_f16((1, 32, 128), 1), k_cache=pkv_inputs.fill_normal_f16(w.pool_shape(), 2),
                v_cache=pkv_inputs.fill_normal_f16(w.pool_shape(), 3), block_table=w.block_table,
                seq_lens=w.seq_lens, Hkv=8, page_size=16, scale=default_scale(128))
    dp = DevProblem(p)
    for hg in (0, 1, 2, 4, 8):
        check(dp, pkv.Policy(tile_tokens=32, num_splits=1, route=pkv.ROUTE_RECT, kernel=kernel, heads_per_cta=hg),
              what="hg%d" % hg)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("Hkv", [8, 4, 16, 32])
@pytest.mark.parametrize("route", [pkv.ROUTE_WORKQUEUE, pkv.ROUTE_RECT])
def test_ragged_split_sweep(kernel, Hkv, route):
    """Ragged rows spanning several tiles and a ragged tail, every split count incl. S > T
    (neutral states), separate and fused merge; G = Hq/Hkv = 4, 8, 2, 1
    (the paper's GQA sweep)."""
    p = make_problem(RAGGED, seed=100 + Hkv, Hkv=Hkv)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for S in (1, 2, 3, 4, 16, 64):
        for mm in (pkv.MERGE_SEPARATE, pkv.MERGE_FUSED):
            pol = pkv.Policy(tile_tokens=32, num_splits=S, route=route, merge_mode=mm, kernel=kernel)
            check(dp, pol, ref, what="S%d mm%d" % (S, mm))
    pol = pkv.Policy(tile_tokens=64, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=2, route=route,
                     kernel=kernel)
    check(dp, pol, ref, what="chunk")


@pytest.mark.parametrize("hg", [1, 2, 4, 8])
@pytest.mark.parametrize("Hkv", [8, 4, 16, 32])
def test_tma_heads_per_cta_variants(hg, Hkv):
    if hg > Hkv:
        pytest.skip("hg > Hkv")
    p = make_problem(RAGGED, seed=300 + Hkv, Hkv=Hkv)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for S, mm in ((1, 0), (5, 0), (5, 1)):
        check(dp, pkv.Policy(tile_tokens=32, num_splits=S, merge_mode=mm, heads_per_cta=hg), ref, what="hg%d S%d" % (hg, S))


@pytest.mark.parametrize("route", [pkv.ROUTE_WORKQUEUE, pkv.ROUTE_RECT])
def test_device_builder_bit_exact(route):
    """pkv_build_workqueue (device) == workqueue oracle: count, order, every field, split_offsets,
    launches and Table-4 counters."""
    rng = np.random.Generator(np.random.PCG64(77))
    cases = [[0], [1], [0, 0], RAGGED, list(rng.integers(0, 70000, size=8)), list(rng.integers(0, 9000, size=128)),
             list(rng.integers(1, 400, size=1500)),
             # very long rows and more shapes for the warp planner (B <= 512)
             [2 ** 24 - 1, 5], [2 ** 24, 7, 100], [2 ** 24 + 17, 2 ** 20, 3], [2 ** 24 - 1] * 3 + [1],
             list(rng.integers(0, 2 ** 22, size=16)), list(rng.integers(0, 300000, size=40)),
             list(rng.integers(0, 5000, size=16)), list(rng.integers(1, 100, size=12)), [65536] * 8,
             list(rng.integers(0, 2 ** 24, size=5))]
    pols = [pkv.Policy(tile_tokens=32, num_splits=20), pkv.Policy(tile_tokens=64, num_splits=0),
            pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=16),
            pkv.Policy(tile_tokens=16, num_splits=256),
            pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0),
            pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=7),
            pkv.Policy(tile_tokens=64, split_mode=pkv.SPLIT_BALANCED, num_splits=12, num_sms=28)]
    for lens in cases:
        lens = np.array(lens, dtype=np.int32)
        for base in pols:
            for Hkv in (8, 4):
                pol = pkv.Policy(**{**base.__dict__, "route": route})
                shape = pkv.Shape(B=len(lens), Hq=32, Hkv=Hkv, max_pages=1, num_pages=1)
                opol = oracle_policy(pol)
                if pol.num_splits == 0 and pol.split_mode == pkv.SPLIT_FIXED_COUNT:
                    opol = wq.Policy(**{**opol.__dict__, "num_sms": sm_count()})
                ref = wq.build_workqueue(list(map(int, lens)), Hkv, opol)
                ws = pkv.alloc_workspace(shape, pol)
                pkv.pkv_build_workqueue(shape, pol, to_dev(lens), ws)
                tasks, offs = pkv.pkv_read_workqueue(shape, pol, ws)
                assert tasks.shape[0] == ref.num_tasks
                assert np.array_equal(tasks, np.array(ref.tasks, dtype=np.int32).reshape(-1, 5))
                assert np.array_equal(offs, np.array(ref.split_offsets, dtype=np.int32))
                c = pkv.pkv_get_counters(shape, pol, ws)
                assert c["tasks"] == ref.num_tasks and c["empty_tasks"] == ref.empty_ctas
                assert c["decode_launches"] == ref.decode_launches and c["merge_launches"] == ref.merge_launches
                assert c["num_splits"] == ref.num_splits and c["chunk_tiles"] == ref.chunk_tiles
                assert c["useful_kv_bytes"] == wq.useful_kv_bytes(lens, Hkv, 128)
                assert c["merge_bytes"] == wq.merge_bytes(ref.num_tasks, 32 // Hkv, 128)


@pytest.mark.parametrize("kernel", KERNELS)
def test_p3_zero_keys_token_counts_exact(kernel):
    """K = 0 => every score is 0, O = mean(V) (closed form) and each partial's l_s is EXACTLY the
    token count of its range (integers < 2^24 are exact in FP32): catches a dropped or duplicated
    token at any N (pin P3)."""
    lens = [4097, 33, 1, 1000]
    p = make_problem(lens, seed=41)
    rng = np.random.Generator(np.random.PCG64(7))
    p.k_cache[...] = 0
    p.v_cache[...] = rng.integers(-8, 9, size=p.v_cache.shape).astype(np.float16)
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=32, num_splits=7, kernel=kernel)
    out, lse, ws = dp.decode(pol)
    ref = oracle_attention(p)
    assert_within_tolerance(out, ref[0])
    q = wq.build_workqueue(lens, 8, oracle_policy(pol))
    m, l, a = read_partials(dp, pol, ws, q.num_tasks)
    for t, (row, kvh, split, tb, te) in enumerate(q.tasks):
        n_i = q.split_offsets[row + 1] - q.split_offsets[row]
        if n_i <= 1:
            continue        # direct output, no partial state
        slot = q.split_offsets[row] * 8 + kvh * n_i + split
        cnt = min(te * 32, lens[row]) - tb * 32
        assert np.all(l[slot] == cnt), (t, l[slot], cnt)
        assert np.all(m[slot] == 0.0)
    assert np.allclose(lse, np.log(np.array(lens, dtype=np.float64))[:, None], atol=1e-5)


@pytest.mark.parametrize("kernel", KERNELS)
def test_p5_dominant_key_at_boundaries(kernel):
    """k_j* = 3 q for the 4 heads sharing... one query head's q: that head's output must be v_j*
    (pin P5).  j* at 0, N-1 and around page / tile / split boundaries."""
    N = 1000
    S = 4
    base = make_problem([N], seed=51)
    c = -(-(-(-N // 32)) // S) * 32      # tokens per split
    spots = sorted({0, 1, 15, 16, 17, 31, 32, 33, c - 1, c, c + 1, 2 * c - 1, 2 * c, N - 2, N - 1})
    for j in spots:
        p = Problem(q=base.q, k_cache=base.k_cache.copy(), v_cache=base.v_cache, block_table=base.block_table,
                    seq_lens=base.seq_lens, Hkv=8, page_size=16, scale=base.scale)
        page, r = token_location(p, 0, j)
        for g in range(8):
            p.k_cache[page, r, g] = (3.0 * p.q[0, g * 4].astype(np.float32)).astype(np.float16)
        dp = DevProblem(p)
        out, _, _ = dp.decode(pkv.Policy(tile_tokens=32, num_splits=S, kernel=kernel))
        for g in range(8):
            want = p.v_cache[page, r, g].astype(np.float64)
            assert np.abs(out[0, g * 4] - want).max() <= 2e-3, (j, g)
        assert_within_tolerance(out, oracle_attention(p)[0], "j=%d" % j)


@pytest.mark.parametrize("kernel", KERNELS)
def test_p2_pool_permutation_bit_identical(kernel):
    p = make_problem([700, 33, 16, 257], seed=21)
    pol = pkv.Policy(tile_tokens=32, num_splits=3, kernel=kernel)
    o1, l1, _ = DevProblem(p).decode(pol)
    o2, l2, _ = DevProblem(permute_pool(p, seed=99)).decode(pol)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)
    o3, l3, _ = DevProblem(p).decode(pol)
    assert np.array_equal(o1, o3) and np.array_equal(l1, l3)      # run-to-run determinism


@pytest.mark.parametrize("kernel", KERNELS)
def test_a10_tail_and_unused_entries_never_contribute(kernel):
    """Tokens past N_i in the last page hold huge values; block-table entries past ceil(N_i/P)
    hold PAD_PAGE: neither may change the result (reading A10)."""
    lens = [45, 100, 17]
    p = make_problem(lens, seed=61, max_pages=40)
    ref = oracle_attention(p)
    for i, N in enumerate(lens):
        page, r = token_location(p, i, N - 1)
        p.k_cache[page, r + 1:] = 60000.0
        p.v_cache[page, r + 1:] = 60000.0
        assert np.all(p.block_table[i, -(-N // 16):] == PAD_PAGE)
    dp = DevProblem(p)
    for S in (1, 3):
        out, _, _ = dp.decode(pkv.Policy(tile_tokens=32, num_splits=S, kernel=kernel))
        assert_within_tolerance(out, ref[0])


@pytest.mark.parametrize("kernel", KERNELS)
def test_paper_layout_strides_reading_a1(kernel):
    """The paper's [page, Hkv, page_size, d] layout through explicit strides."""
    p = make_problem([300, 19], seed=31)
    ref = oracle_attention(p)
    k_hnd = to_dev(np.ascontiguousarray(p.k_cache.transpose(0, 2, 1, 3)))
    v_hnd = to_dev(np.ascontiguousarray(p.v_cache.transpose(0, 2, 1, 3)))
    dp = DevProblem(p, kv_strides=(8 * 16 * 128, 128, 16 * 128), k_dev=k_hnd, v_dev=v_hnd)
    for S in (1, 4):
        out, _, _ = dp.decode(pkv.Policy(tile_tokens=32, num_splits=S, kernel=kernel))
        assert_within_tolerance(out, ref[0])


def test_n1_bit_exact_and_scale_argument():
    """N = 1 => O = v_0 bit-exactly in FP16 (pin P6); an explicit scale is honoured."""
    p = make_problem([1, 1, 1], seed=71)
    dp = DevProblem(p)
    for kernel in KERNELS:
        out, lse, _ = dp.decode(pkv.Policy(num_splits=1, kernel=kernel))
        for i in range(3):
            page, r = token_location(p, i, 0)
            want = np.repeat(p.v_cache[page, r].astype(np.float64), 4, axis=0)
            assert np.array_equal(out[i], want)
    p2 = make_problem([90], seed=72)
    p2.scale = 0.25
    dp2 = DevProblem(p2)
    out, lse, _ = dp2.decode(pkv.Policy(num_splits=2))
    ref = oracle_attention(p2)
    assert_within_tolerance(out, ref[0])
    out0, _, _ = dp2.decode(pkv.Policy(num_splits=2), scale=0.0)     # <= 0 means 1/sqrt(d)
    p2.scale = default_scale(128)
    assert_within_tolerance(out0, oracle_attention(p2)[0])


def test_pkv_merge_standalone_vs_oracle():
    """pkv_merge on caller-provided states (public partial format) == oracle merge,
    including neutral states and a row without any state."""
    rng = np.random.Generator(np.random.PCG64(5))
    Hkv, G, d = 8, 4, 128
    n = [3, 0, 1, 17]
    offs = np.concatenate([[0], np.cumsum(n)]).astype(np.int32)
    slots = int(offs[-1]) * Hkv
    m = rng.normal(0, 3, size=(slots, G)).astype(np.float32)
    l = rng.uniform(0.5, 50, size=(slots, G)).astype(np.float32)
    a = rng.normal(0, 4, size=(slots, G, d)).astype(np.float32)
    m[1], l[1], a[1] = -np.inf, 0.0, 0.0                 # a neutral state inside row 0
    shape = pkv.Shape(B=len(n), Hq=32, Hkv=Hkv)
    out = torch.full((len(n), 32, d), float("nan"), dtype=torch.float16, device="cuda")
    lse = torch.full((len(n), 32), float("nan"), dtype=torch.float32, device="cuda")
    pkv.pkv_merge(shape, to_dev(m), to_dev(l), to_dev(a), to_dev(offs), out, lse)
    torch.cuda.synchronize()
    out, lse = out.cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64)
    for i, n_i in enumerate(n):
        for g in range(Hkv):
            b = int(offs[i]) * Hkv + g * n_i
            for hh in range(G):
                o_ref, lse_ref = pkv_oracle.merge(m[b:b + n_i, hh], l[b:b + n_i, hh], a[b:b + n_i, hh])
                h = g * G + hh
                if n_i == 0:
                    assert np.all(out[i, h] == 0) and np.isneginf(lse[i, h])
                else:
                    assert np.abs(out[i, h] - o_ref).max() <= 2e-3 * max(1.0, np.abs(o_ref).max())
                    assert abs(lse[i, h] - lse_ref) <= 1e-4


def test_partial_states_match_oracle_split_states():
    """GPU partial states vs the oracle's split form through the invariant pair
    LSE_s = m_s + log l_s, O_s = a_s / l_s (reading A11)."""
    lens = [1500, 64, 333]
    p = make_problem(lens, seed=81)
    dp = DevProblem(p)
    for kernel in KERNELS:
        pol = pkv.Policy(tile_tokens=32, num_splits=5, kernel=kernel)
        _, _, ws = dp.decode(pol)
        q = wq.build_workqueue(lens, 8, oracle_policy(pol))
        tasks = np.array(q.tasks, dtype=np.int32)
        rm, rl, ra = pkv_oracle.split_states(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens, tasks, Hkv=8,
                                             page_size=16, tile_tokens=32, scale=p.scale)
        m, l, a = read_partials(dp, pol, ws, q.num_tasks)
        # canonical order == slot order (reading A8)
        assert np.abs((m + np.log(l)) - (rm + np.log(rl))).max() <= 1e-4
        assert np.abs(a / l[..., None] - ra / rl[..., None]).max() <= 2e-3


def test_decode_host_entry_point():
    """pkv_decode_host: host planning + one H2D image + decode + merge + D2H;
    launch counts equal the oracle's (reading A13)."""
    lens = [1500, 64, 0, 333]
    p = make_problem(lens, seed=91)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(num_splits=6), pkv.Policy(num_splits=1), pkv.Policy(num_splits=6, merge_mode=pkv.MERGE_FUSED),
                pkv.Policy(num_splits=6, route=pkv.ROUTE_RECT, kernel=pkv.KERNEL_SIMT)):
        nb = pkv.pkv_host_scratch_bytes(dp.shape, pol)
        staging = torch.zeros(nb, dtype=torch.uint8).pin_memory()
        scratch = torch.empty(nb, dtype=torch.uint8, device="cuda")
        ws = pkv.alloc_workspace(dp.shape, pol)
        out = np.full((p.B, p.Hq, p.d), np.nan, dtype=np.float16)
        c = pkv.pkv_decode_host(dp.shape, pol, p.q, dp.k, dp.v, p.block_table, p.seq_lens, out, p.scale, staging,
                                scratch, ws)
        assert_within_tolerance(out.astype(np.float64), ref[0])
        q = wq.build_workqueue(lens, 8, oracle_policy(pol))
        assert c["tasks"] == q.num_tasks
        assert c["decode_launches"] == q.decode_launches and c["merge_launches"] == q.merge_launches
        assert c["d2h_bytes"] == out.nbytes and c["h2d_bytes"] > p.q.nbytes
        # pinned out_host: the kernels write the result straight into host memory (zero copy)
        out_pin = torch.full((p.B, p.Hq, p.d), float("nan"), dtype=torch.float16).pin_memory()
        pkv.pkv_decode_host(dp.shape, pol, p.q, dp.k, dp.v, p.block_table, p.seq_lens, out_pin.data_ptr(), p.scale,
                            staging, scratch, ws)
        assert np.array_equal(out_pin.numpy(), out)
    # every row empty: no launch at all, out = 0
    p0 = make_problem([0, 0], seed=92)
    dp0 = DevProblem(p0)
    pol = pkv.Policy(num_splits=2)
    nb = pkv.pkv_host_scratch_bytes(dp0.shape, pol)
    out = np.full((2, 32, 128), np.nan, dtype=np.float16)
    c = pkv.pkv_decode_host(dp0.shape, pol, p0.q, dp0.k, dp0.v, p0.block_table, p0.seq_lens, out, p0.scale,
                            torch.zeros(nb, dtype=torch.uint8).pin_memory(),
                            torch.empty(nb, dtype=torch.uint8, device="cuda"), pkv.alloc_workspace(dp0.shape, pol))
    assert np.all(out == 0) and c["decode_launches"] == 0 and c["merge_launches"] == 0


@pytest.mark.parametrize("mode", [pkv.SPLIT_FIXED_COUNT, pkv.SPLIT_AUTO])
def test_decode_host_serving_loop_uploads_only_what_changed(mode):
    """A serving loop through pkv_decode_host on one (staging, scratch) pair: lengths grow across
    page boundaries, one request is replaced by another (its whole table row changes), one finishes
    (N = 0).  Every step matches the oracle and leaves the oracle's queue in the workspace; of the
    block table only changed rows are uploaded (h2d_bytes); PKV_SPLIT_AUTO re-plans per step."""
    lens = np.array([1500, 62, 4000, 333], dtype=np.int32)
    p = make_problem(list(lens + 40), seed=93)
    p2 = make_problem(list(lens + 40), seed=94)              # other page assignment, same pool size
    assert p2.k_cache.shape == p.k_cache.shape
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=32, split_mode=mode, num_splits=5 if mode == pkv.SPLIT_FIXED_COUNT else 0)
    nb = pkv.pkv_host_scratch_bytes(dp.shape, pol)
    staging = torch.zeros(nb, dtype=torch.uint8).pin_memory()
    scratch = torch.empty(nb, dtype=torch.uint8, device="cuda")
    ws = pkv.alloc_workspace(dp.shape, pol)
    out = torch.full((p.B, p.Hq, p.d), float("nan"), dtype=torch.float16).pin_memory()
    table = p.block_table.copy()
    row_bytes = 4 * table.shape[1]
    base = p.q.nbytes + 256                                  # seq_lens (padded to 256) + q in one copy
    shadow, seen = np.zeros_like(table), []
    for t in range(8):
        cur = (lens + t).astype(np.int32)
        if t >= 3:
            table[1] = p2.block_table[1] % p.k_cache.shape[0]          # row 1 now holds another request
        if t >= 5:
            cur[3] = 0
        p.seq_lens, p.block_table = cur, table
        c = pkv.pkv_decode_host(dp.shape, pol, p.q, dp.k, dp.v, table, cur, out.data_ptr(), p.scale, staging, scratch, ws)
        ref, _ = oracle_attention(p)
        assert_within_tolerance(out.numpy().astype(np.float64), ref, "step %d" % t)
        # rows whose used entries differ from what the device holds (all of them at step 0)
        nchanged = 0
        for i in range(p.B):
            used = -(-int(cur[i]) // 16)
            if used and (t == 0 or not np.array_equal(table[i, :used], shadow[i, :used])):
                shadow[i, :used] = table[i, :used]
                nchanged += 1
        assert c["h2d_bytes"] == base + nchanged * row_bytes, (t, nchanged)
        seen.append(nchanged)
        assert c["h2d_bytes"] <= base + 4 * row_bytes and c["d2h_bytes"] == out.numel() * 2
        if mode == pkv.SPLIT_FIXED_COUNT:
            q = wq.build_workqueue(list(cur), 8, oracle_policy(pol))
            assert c["tasks"] == q.num_tasks and c["decode_launches"] == q.decode_launches and c["merge_launches"] == q.merge_launches
            tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
            assert tasks.tolist() == [list(x) for x in q.tasks] and offs.tolist() == q.split_offsets
    assert seen[0] == 4 and 0 in seen and max(seen[1:]) <= 2
    # steady state: nothing but lengths and q goes up
    c = pkv.pkv_decode_host(dp.shape, pol, p.q, dp.k, dp.v, table, cur, out.data_ptr(), p.scale, staging, scratch, ws)
    assert c["h2d_bytes"] == base
    # the prepared call (pkv.HostDecoder): same result bit for bit, same bytes
    want = out.numpy().copy()
    qpin, lpin = torch.from_numpy(p.q.copy()).pin_memory(), torch.from_numpy(cur.copy()).pin_memory()
    out.fill_(float("nan"))
    dec = pkv.HostDecoder(dp.shape, pol, dp.k, dp.v, staging, scratch, ws, p.scale)
    for _ in range(2):
        dec(qpin.data_ptr(), table.ctypes.data, lpin.data_ptr(), out.data_ptr())
    assert np.array_equal(out.numpy(), want)
    assert dec.counters["h2d_bytes"] == base


@pytest.mark.parametrize("mm", [pkv.MERGE_SEPARATE, pkv.MERGE_FUSED])
def test_cuda_graph_replay_with_growing_lengths(mm):
    """{device builder, decode, merge} captured once and replayed while seq_lens grows in place
    (north_star (e)): the task count changes between replays, the graph does not."""
    lens = np.array([60, 1000, 31, 257], dtype=np.int32)
    steps = 40
    p = make_problem(lens, seed=95, reserve_extra=steps)
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=32, num_splits=4, merge_mode=mm)
    ws = pkv.alloc_workspace(dp.shape, pol)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        pkv.pkv_decode(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, dp.out, dp.lse, scale=p.scale, workspace=ws,
                       stream=s)       # warm-up outside capture (sets function attributes)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            pkv.pkv_decode(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, dp.out, dp.lse, scale=p.scale,
                           workspace=ws, stream=torch.cuda.current_stream())
    for step in range(steps):
        dp.sl.copy_(torch.from_numpy(lens + step))
        dp.out.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        if step % 13 == 0 or step == steps - 1:
            p.seq_lens = (lens + step).astype(np.int32)
            assert_within_tolerance(dp.out.cpu().numpy().astype(np.float64), oracle_attention(p)[0], "step %d" % step)
            tasks, _ = pkv.pkv_read_workqueue(dp.shape, pol, ws)
            assert tasks.shape[0] == wq.build_workqueue(list(lens + step), 8, oracle_policy(pol)).num_tasks


@pytest.mark.parametrize("Hkv", [8, 4])
@pytest.mark.parametrize("hg", [1, 2, 4, 8])
def test_many_units_per_cta_odd_page_counts(hg, Hkv):
    """More work units than SMs, rows with odd page counts: every persistent CTA walks several
    units, so its page ring wraps across unit boundaries with every residue of the page sequence
    number (the stage-ownership rule of the multi-producer ring)."""
    if hg > Hkv:
        pytest.skip("hg > Hkv")
    rng = np.random.Generator(np.random.PCG64(1234 + hg))
    lens = rng.integers(1, 1500, size=96).astype(np.int32)
    lens[::7] = rng.integers(1, 40, size=len(lens[::7]))          # some one- and two-page rows
    p = make_problem(list(lens), seed=400 + hg, Hkv=Hkv)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(tile_tokens=32, num_splits=1), pkv.Policy(tile_tokens=16, num_splits=3),
                pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=5,
                           merge_mode=pkv.MERGE_FUSED)):
        pol.heads_per_cta = hg
        for _ in range(2):          # twice: the dynamic unit counter must have re-armed itself
            check(dp, pol, ref, what="hg%d %s" % (hg, pol))


@pytest.mark.parametrize("Hkv", [8, 4])
@pytest.mark.parametrize("hg", [1, 2, 4, 8])
def test_long_units_ring_wraps_many_times(hg, Hkv):
    """Units of 16 pages and more on rings of 3..24 stages, several units per CTA, with several
    compute warps per head (8 / hg) and several producers: a stage must be filled and consumed by
    the same warps in every one of its phases; a warp that skips a
    phase of a stage can pass the parity wait of the next phase early and read a stale page."""
    if hg > Hkv:
        pytest.skip("hg > Hkv")
    rng = np.random.Generator(np.random.PCG64(77 + hg))
    lens = rng.integers(1, 3000, size=128).astype(np.int32)
    p = make_problem(list(lens), seed=500 + hg, Hkv=Hkv)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=8),
                pkv.Policy(tile_tokens=32, num_splits=1), pkv.Policy(tile_tokens=32, num_splits=4)):
        pol.heads_per_cta = hg
        for _ in range(3):
            check(dp, pol, ref, what="hg%d %s" % (hg, pol))


def test_pdl_off_matches_pdl_on_bitwise():
    """Programmatic dependent launch only changes when kernels start, never what they compute."""
    p = make_problem([700, 33, 16, 257, 0, 2000], seed=23)
    pol = pkv.Policy(tile_tokens=32, num_splits=5)
    dp = DevProblem(p)
    o1, l1, _ = dp.decode(pol)
    o2, l2, _ = dp.decode(dataclasses.replace(pol, flags=pkv.FLAG_NO_PDL))
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)
    assert_within_tolerance(o1, oracle_attention(p)[0])


@pytest.mark.parametrize("route", [pkv.ROUTE_WORKQUEUE, pkv.ROUTE_RECT])
def test_fused_build_queue_bit_exact_and_same_output(route):
    """pkv_decode's fused build (the TMA kernel derives the queue from seq_lens itself) leaves the
    same queue in the workspace as the builder kernel and the oracle: count, order,
    every field, split_offsets, counters; outputs are bitwise equal with the builder kernel's."""
    lens = [700, 0, 33, 16, 257, 1, 2000, 31, 64, 65]
    p = make_problem(lens, seed=29)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    pols = [pkv.Policy(tile_tokens=32, num_splits=5, route=route),
            pkv.Policy(tile_tokens=16, num_splits=0, route=route),
            pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=3, route=route),
            pkv.Policy(tile_tokens=32, num_splits=7, route=route, merge_mode=pkv.MERGE_FUSED),
            pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, route=route),
            pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=5, route=route)]
    for pol in pols:
        opol = oracle_policy(pol)
        if pol.num_splits == 0 and pol.split_mode == pkv.SPLIT_FIXED_COUNT:
            opol = wq.Policy(**{**opol.__dict__, "num_sms": sm_count()})
        want = wq.build_workqueue(lens, 8, opol)
        outs = []
        for fused in (True, False):
            pol = dataclasses.replace(pol, flags=0 if fused else pkv.FLAG_SEPARATE_BUILD)
            out, lse, ws, _ = check(dp, pol, ref, what="fused=%s %s" % (fused, pol))
            outs.append((out, lse))
            tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
            assert np.array_equal(tasks, np.array(want.tasks, dtype=np.int32).reshape(-1, 5)), (fused, pol)
            assert np.array_equal(offs, np.array(want.split_offsets, dtype=np.int32))
            c = pkv.pkv_get_counters(dp.shape, pol, ws)
            assert c["tasks"] == want.num_tasks and c["empty_tasks"] == want.empty_ctas
            assert c["decode_launches"] == want.decode_launches and c["merge_launches"] == want.merge_launches
            assert c["build_launches"] == (0 if fused else 1) and c["chunk_tiles"] == want.chunk_tiles
        assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


@pytest.mark.parametrize("Hkv", [8, 4])
@pytest.mark.parametrize("kernel", KERNELS)
def test_balanced_policy_parity_single_wave_and_many_waves(kernel, Hkv):
    """BALANCED split policy (A21) end to end: a ragged batch whose chunk comes from
    the single-wave search (device SM count) and one forced into the many-wave regime
    (num_sms = 3); tasks bit-exact vs the oracle, outputs within tolerance."""
    lens = [9000, 40, 1300, 0, 517, 4097, 16, 2222]
    p = make_problem(lens, seed=41, Hkv=Hkv)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, kernel=kernel),
                pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=3, kernel=kernel),
                pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=3, kernel=kernel,
                           merge_mode=pkv.MERGE_FUSED)):
        out, lse, ws, _ = check(dp, pol, ref, what=str(pol))
        want = wq.build_workqueue(lens, Hkv, oracle_policy(pol))
        tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
        assert np.array_equal(tasks, np.array(want.tasks, dtype=np.int32).reshape(-1, 5)), pol
        assert np.array_equal(offs, np.array(want.split_offsets, dtype=np.int32))
        assert pkv.pkv_get_counters(dp.shape, pol, ws)["chunk_tiles"] == want.chunk_tiles


def test_stage_release_waits_for_the_last_ldmatrix():
    """Regression: a compute warp's mbarrier arrive on a stage's
    `empty` barrier was scheduled right behind the ISSUE of its last ldmatrix and could overtake
    it while the planner warp's queue stores backed up the SM's memory pipe; the producer then
    refilled the stage under the load.  K = 0 makes every token's weight exactly 1, V rows are
    one-hot tags of the token index mod 128, so out * N counts the tokens seen per tag: any
    token read from another page shows up as a count that is off by one (it was 1..4 tags in
    about 2 % of the launches, always in channels 112..127 -- the last ldmatrix)."""
    rng = np.random.Generator(np.random.PCG64(10002))
    B = 200
    lens = rng.integers(1, 3000, size=B).astype(np.int32)
    p = make_problem(list(lens), seed=502)
    p.k_cache[:] = 0
    p.v_cache[:] = 0
    exp = np.zeros((B, 128))
    for i in range(B):
        j = np.arange(lens[i])
        p.v_cache[p.block_table[i, j // 16], j % 16, :, j % 128] = 1.0
        exp[i] = np.bincount(j % 128, minlength=128)
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=2)
    ws = pkv.alloc_workspace(dp.shape, pol)
    for rep in range(120):
        out, lse, _ = dp.decode(pol, ws=ws)
        cnt = out * lens[:, None, None].astype(np.float64)
        assert np.abs(cnt - exp[:, None, :]).max() < 0.3, "launch %d: a token was read from another page" % rep
        assert np.abs(lse - np.log(lens)[:, None]).max() < 1e-5


def _compact_rows(w, k_dev, v_dev, rows, lens):
    """Host copy of the pages of `rows` only (compact pool + identity tables), for the oracle."""
    P = w.page_size
    tables, ks, vs, base = [], [], [], 0
    width = max(-(-int(lens[i]) // P) for i in rows)
    for i in rows:
        npg = -(-int(lens[i]) // P)
        pages = torch.from_numpy(w.block_table[i, :npg].astype(np.int64)).cuda()
        ks.append(k_dev[pages].cpu().numpy())
        vs.append(v_dev[pages].cpu().numpy())
        t = np.full(width, pkv_inputs.PAD_PAGE, dtype=np.int32)
        t[:npg] = np.arange(base, base + npg, dtype=np.int32)
        tables.append(t)
        base += npg
    return np.concatenate(ks), np.concatenate(vs), np.stack(tables)


FULL_SIZE_CASES = ["config2", "config3", "config3_rect", "config3_fused", "config4", "config4_b4", "config5",
                   "config5_hkv4"]


@pytest.mark.parametrize("name", FULL_SIZE_CASES)
def test_full_size_configs_in_the_bench_configuration(name):
    """BASELINE.json's full sizes with the policies bench.py times (config 2: the sweep's
    FIXED_COUNT S=16 and BALANCED; others: BALANCED, page-granular tiles), seeded device pools as in
    bench.py.  Rows are checked one by one against the oracle on a host copy of their pages (all
    rows up to B = 8; config 5: the shortest, the longest and two more of the 128); the task list of
    the whole batch is bit-exact; token coverage at full size is pinned by lse = log-sum-exp."""
    import pkv_inputs as pi
    from oracle import pkv_oracle
    seed = pi.REPORT_SEEDS[0]
    w = {"config2": pi.config2, "config3": pi.config3, "config3_rect": pi.config3, "config3_fused": pi.config3,
         "config4": pi.config4, "config4_b4": pi.config4_b4, "config5": pi.config5,
         "config5_hkv4": lambda s_: pi.config5(s_, Hkv=4)}[name](seed)
    dev = torch.device("cuda", 0)
    q = pi.fill_pool_torch((w.B, w.Hq, w.d), 11, dev)
    k = pi.fill_pool_torch(w.pool_shape(), 12, dev)
    v = pi.fill_pool_torch(w.pool_shape(), 13, dev)
    bt = torch.from_numpy(w.block_table).to(dev)
    lens = w.seq_lens_at(min(w.steps, 7)).astype(np.int32)
    sl = torch.from_numpy(lens).to(dev)
    shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, max_pages=w.max_pages, num_pages=w.num_pages)
    pols = [pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0)]
    # what bench.py times: the cost model's choice for these lengths (pkv_choose_policy, default constants)
    auto, _ = pkv.pkv_choose_policy(shape, lens, pkv.pkv_default_cost_model(sm_count()),
                                    pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_AUTO, num_splits=0))
    pols.append(auto)
    if name == "config2":
        pols.append(pkv.Policy(tile_tokens=32, num_splits=16))
        pols.append(pkv.Policy(tile_tokens=32, num_splits=16, merge_mode=pkv.MERGE_FUSED))
        pols.append(pkv.Policy(tile_tokens=32, num_splits=128))          # channel-sliced merge, 128 whole-page units
    if name == "config3_rect":      # BASELINE.json configs[2]: the rectangular (B, Hkv, S) grid
        pols = [pkv.Policy(tile_tokens=32, num_splits=20, route=pkv.ROUTE_RECT),
                pkv.Policy(tile_tokens=32, num_splits=20, route=pkv.ROUTE_WORKQUEUE)]
    if name == "config3_fused":     # fused last-CTA merge at full size
        pols = [pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, merge_mode=pkv.MERGE_FUSED),
                pkv.Policy(tile_tokens=32, num_splits=20, merge_mode=pkv.MERGE_FUSED)]
    if w.B <= 8:
        rows = list(range(w.B))
    else:           # config 5: shortest, longest and 16 seeded rows of the 128
        pick = np.random.Generator(np.random.PCG64(seed)).choice(w.B, size=16, replace=False)
        rows = sorted({int(np.argmin(lens)), int(np.argmax(lens))} | {int(x) for x in pick})
    kc, vc, tc = _compact_rows(w, k, v, rows, lens)
    scale = default_scale(w.d)
    ref, ref_lse = pkv_oracle.attention(np.ascontiguousarray(q.cpu().numpy()[rows]), kc, vc, tc,
                                        np.ascontiguousarray(lens[rows]), Hkv=w.Hkv, page_size=w.page_size, scale=scale)
    for pol in pols:
        out = torch.full((w.B, w.Hq, w.d), float("nan"), dtype=torch.float16, device=dev)
        lse = torch.full((w.B, w.Hq), float("nan"), dtype=torch.float32, device=dev)
        ws = pkv.alloc_workspace(shape, pol)
        pkv.pkv_decode(shape, pol, q, k, v, bt, sl, out, lse, scale=scale, workspace=ws)
        torch.cuda.synchronize()
        got = out.cpu().numpy().astype(np.float64)
        assert not np.isnan(got).any()
        assert_within_tolerance(got[rows], ref, "%s %s" % (name, pol))
        assert np.abs(lse.cpu().numpy().astype(np.float64)[rows] - ref_lse).max() <= 2e-3
        want = wq.build_workqueue([int(x) for x in lens], w.Hkv, oracle_policy(pol))
        tasks, offs = pkv.pkv_read_workqueue(shape, pol, ws)
        assert np.array_equal(tasks, np.array(want.tasks, dtype=np.int32).reshape(-1, 5))
        assert np.array_equal(offs, np.array(want.split_offsets, dtype=np.int32))


@pytest.mark.parametrize("mode", [pkv.SPLIT_FIXED_COUNT, pkv.SPLIT_BALANCED])
def test_speculative_plan_is_discarded_when_lengths_changed(mode):
    """The TMA kernel plans from seq_lens before its dependency wait and validates the lengths
    afterwards.  With the test hook every launch behaves as if the
    kernel right before it had rewritten seq_lens: a deliberately wrong speculative plan is left
    behind and the kernel must plan again.  Same queue, bitwise the same output as without it."""
    lens = [9000, 40, 1300, 0, 517, 4097, 16, 2222]
    p = make_problem(lens, seed=43)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    pol = pkv.Policy(tile_tokens=16, split_mode=mode, num_splits=0 if mode == pkv.SPLIT_BALANCED else 6)
    o1, l1, ws1, _ = check(dp, pol, ref)
    o2, l2, ws2, _ = check(dp, dataclasses.replace(pol, flags=pkv.FLAG_TEST_REPLAN), ref)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)
    t1, f1 = pkv.pkv_read_workqueue(dp.shape, pol, ws1)
    t2, f2 = pkv.pkv_read_workqueue(dp.shape, pol, ws2)
    assert np.array_equal(t1, t2) and np.array_equal(f1, f2)
    # seq_lens rewritten on the device right before the call (stream order): the new lengths count
    new = np.array([100, 40, 1300, 0, 517, 33, 16, 2000], dtype=np.int32)     # within the reserved pages
    dp.sl.copy_(to_dev(new))
    p.seq_lens = new
    check(dp, pol, oracle_attention(p))


@pytest.mark.parametrize("variant", ["fp8", "append", "buckets"])
@pytest.mark.parametrize("name", ["config2", "config3"])
def test_full_size_round2_routes(name, variant):
    """BASELINE.json's config 2 and 3 at full size through the round-2 paths as bench.py times them
    (cost-model policy): FP8 caches against the FP8 oracle, the fused KV-append + RoPE step against the
    append oracle (outputs and the pool bytes of the new tokens), exact length buckets against the
    FP16 oracle.  Every row of the batch is checked."""
    import pkv_inputs as pi
    from oracle import append_oracle, pkv_oracle
    seed = pi.REPORT_SEEDS[0]
    w = {"config2": pi.config2, "config3": pi.config3}[name](seed)
    dev = torch.device("cuda", 0)
    q = pi.fill_pool_torch((w.B, w.Hq, w.d), 21, dev)
    k = pi.fill_pool_torch(w.pool_shape(), 22, dev)
    v = pi.fill_pool_torch(w.pool_shape(), 23, dev)
    bt = torch.from_numpy(w.block_table).to(dev)
    lens = w.seq_lens_at(min(w.steps, 5)).astype(np.int32)
    sl = torch.from_numpy(lens).to(dev)
    rows = list(range(w.B))
    scale = default_scale(w.d)
    qh = np.ascontiguousarray(q.cpu().numpy())
    out = torch.full((w.B, w.Hq, w.d), float("nan"), dtype=torch.float16, device=dev)
    lse = torch.full((w.B, w.Hq), float("nan"), dtype=torch.float32, device=dev)
    base = pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_AUTO, num_splits=0)
    if variant == "fp8":
        sc = torch.full((w.Hkv,), 1.0 / 32.0, dtype=torch.float32, device=dev)
        k = (k.float() * 32.0).to(torch.float8_e4m3fn).view(torch.uint8)
        v = (v.float() * 32.0).to(torch.float8_e4m3fn).view(torch.uint8)
        shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, max_pages=w.max_pages, num_pages=w.num_pages, kv_dtype=pkv.KV_E4M3,
                          k_scale=sc, v_scale=sc)
        pol, _ = pkv.pkv_choose_policy(shape, lens, pkv.pkv_default_cost_model(sm_count()), base)
        kc, vc, tc = _compact_rows(w, k, v, rows, lens)
        s64 = np.full(w.Hkv, 1.0 / 32.0)
        ref, ref_lse = pkv_oracle.attention_fp8(qh, kc, vc, s64, s64, tc, lens, Hkv=w.Hkv, page_size=w.page_size, scale=scale)
        pkv.pkv_decode(shape, pol, q, k, v, bt, sl, out, lse, scale=scale, workspace=pkv.alloc_workspace(shape, pol))
    else:
        shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, max_pages=w.max_pages, num_pages=w.num_pages)
        pol, _ = pkv.pkv_choose_policy(shape, lens, pkv.pkv_default_cost_model(sm_count()), base)
        kc, vc, tc = _compact_rows(w, k, v, rows, lens)
        if variant == "append":
            kn = pi.fill_pool_torch((w.B, w.Hkv, w.d), 24, dev)
            vn = pi.fill_pool_torch((w.B, w.Hkv, w.d), 25, dev)
            npos = int(lens.max()) + 1
            inv = 10000.0 ** (-np.arange(0, w.d // 2, dtype=np.float64) * 2.0 / w.d)
            ang = np.arange(npos, dtype=np.float64)[:, None] * inv[None, :]
            cos, sin = np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)
            ref, ref_lse, k2, v2 = append_oracle.append_and_attend(qh, kc, vc, kn.cpu().numpy(), vn.cpu().numpy(), tc, lens, cos, sin,
                                                                   Hkv=w.Hkv, page_size=w.page_size, scale=scale)
            app = pkv.Append(k_new=kn, v_new=vn, rope_cos=torch.from_numpy(cos).to(dev), rope_sin=torch.from_numpy(sin).to(dev),
                             rope_positions=npos)
            pkv.pkv_decode_append(shape, pol, q, k, v, bt, sl, None, app, out, lse, scale=scale,
                                  workspace=pkv.alloc_workspace(shape, pol))
            torch.cuda.synchronize()
            kc_after, vc_after, _ = _compact_rows(w, k, v, rows, lens)
            assert np.array_equal(kc_after.view(np.uint16), k2.view(np.uint16))
            assert np.array_equal(vc_after.view(np.uint16), v2.view(np.uint16))
        else:
            ref, ref_lse = pkv_oracle.attention(qh, kc, vc, tc, lens, Hkv=w.Hkv, page_size=w.page_size, scale=scale)
            pol = pkv.Policy(tile_tokens=32, num_splits=32, route=pkv.ROUTE_RECT)
            index, offs, _ = pkv.pkv_plan_buckets_host(lens, 1)
            pkv.pkv_decode_buckets(shape, pol, q, k, v, bt, sl, torch.from_numpy(index).to(dev), offs, out, lse, scale=scale,
                                   workspace=pkv.alloc_workspace(shape, pol))
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    assert not np.isnan(got).any()
    assert_within_tolerance(got, ref, "%s %s %s" % (name, variant, pol))
    assert np.abs(lse.cpu().numpy().astype(np.float64) - ref_lse).max() <= 2e-3
