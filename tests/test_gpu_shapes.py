"""GPU parity for the shapes of SURVEY.md sec. 8(f) f2: page sizes
32 and 64 ("heterogeneous page sizes"), G = Hq / Hkv = 16, head dimensions 64 and 256.  The oracle
takes any shape (tests/test_oracle_pins.py, P1 on other shapes); here the CUDA path is compared
with it element by element, token coverage is pinned by the K = 0 counting test, and page / tile /
split boundaries by the dominant key."""
import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
from gpu_helpers import DevProblem, oracle_attention, oracle_policy, read_partials
from helpers import assert_within_tolerance, make_problem, token_location, Problem
from oracle import workqueue_oracle as wq

pytestmark = pytest.mark.gpu

KERNELS = [pkv.KERNEL_TMA_MMA, pkv.KERNEL_SIMT]
RAGGED = [1, 2, 15, 16, 17, 31, 32, 33, 63, 64, 65, 100, 0, 257, 700, 4099]


def _check(dp, pol, ref, what):
    out, lse, ws = dp.decode(pol)
    assert not np.isnan(out).any(), what
    assert_within_tolerance(out, ref[0], what)
    fin = np.isfinite(ref[1])
    assert np.array_equal(np.isneginf(lse), np.isneginf(ref[1])), what
    assert np.abs(lse[fin] - ref[1][fin]).max(initial=0.0) <= 2e-3, what
    return out, lse, ws


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("P", [32, 64])
@pytest.mark.parametrize("Hkv", [8, 4])
def test_page_sizes_ragged_sweep(kernel, P, Hkv):
    p = make_problem(RAGGED, seed=600 + P + Hkv, Hkv=Hkv, page_size=P)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(tile_tokens=P, num_splits=1, kernel=kernel),
                pkv.Policy(tile_tokens=P, num_splits=3, kernel=kernel),
                pkv.Policy(tile_tokens=2 * P, num_splits=5, kernel=kernel, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT),
                pkv.Policy(tile_tokens=P, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=20, kernel=kernel),
                pkv.Policy(tile_tokens=P, num_splits=4, kernel=kernel, heads_per_cta=2),
                pkv.Policy(tile_tokens=P, num_splits=2, kernel=kernel, heads_per_cta=1, prefetch_kb=64)):
        _, _, ws = _check(dp, pol, ref, "P%d %s" % (P, pol))
        tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
        want = wq.build_workqueue(RAGGED, Hkv, oracle_policy(pol))
        assert tasks.tolist() == [list(t) for t in want.tasks] and offs.tolist() == want.split_offsets


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("P", [32, 64])
def test_page_sizes_token_counts_exact_and_dominant_key(kernel, P):
    """Pins P3 and P5 at page sizes 32 / 64: with K = 0 every partial's l_s is exactly its token
    count; a dominant key at every block (16 tokens), page, tile and split boundary +-1 returns
    exactly that token's V."""
    lens = [4097, 33, 1, 1000]
    p = make_problem(lens, seed=41 + P, page_size=P)
    rng = np.random.Generator(np.random.PCG64(7))
    p.k_cache[...] = 0
    p.v_cache[...] = rng.integers(-8, 9, size=p.v_cache.shape).astype(np.float16)
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=P, num_splits=7, kernel=kernel)
    out, lse, ws = dp.decode(pol)
    assert_within_tolerance(out, oracle_attention(p)[0])
    q = wq.build_workqueue(lens, 8, oracle_policy(pol))
    m, l, a = read_partials(dp, pol, ws, q.num_tasks)
    for (row, kvh, split, tb, te) in q.tasks:
        n_i = q.split_offsets[row + 1] - q.split_offsets[row]
        if n_i > 1:
            slot = q.split_offsets[row] * 8 + kvh * n_i + split
            assert np.all(l[slot] == min(te * P, lens[row]) - tb * P) and np.all(m[slot] == 0.0)
    N, S = 1000, 3
    base = make_problem([N], seed=51 + P, page_size=P)
    c = -(-(-(-N // P)) // S) * P
    spots = sorted({0, 15, 16, 17, 31, 32, 33, 47, 48, 63, 64, 65, c - 1, c, c + 1, 2 * c - 1, 2 * c, N - 2, N - 1})
    for j in spots:
        pj = Problem(q=base.q, k_cache=base.k_cache.copy(), v_cache=base.v_cache, block_table=base.block_table,
                     seq_lens=base.seq_lens, Hkv=8, page_size=P, scale=base.scale)
        page, r = token_location(pj, 0, j)
        for g in range(8):
            pj.k_cache[page, r, g] = (3.0 * pj.q[0, g * 4].astype(np.float32)).astype(np.float16)
        out, _, _ = DevProblem(pj).decode(pkv.Policy(tile_tokens=P, num_splits=S, kernel=kernel))
        for g in range(8):
            assert np.abs(out[0, g * 4] - pj.v_cache[page, r, g].astype(np.float64)).max() <= 2e-3, (j, g)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("Hq,Hkv", [(32, 2), (64, 4), (128, 8)])
def test_g16_ragged_sweep(kernel, Hq, Hkv):
    """G = Hq / Hkv = 16 ("G=1 and G=8 ... until separate mappings are
    implemented"): two blocks of 8 query heads per KV head share each streamed K/V stage.  Every
    heads-per-CTA variant, both routes, separate and fused merge; queue bit-exact."""
    p = make_problem(RAGGED, seed=700 + Hkv, Hq=Hq, Hkv=Hkv)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    hgs = [h for h in (0, 1, 2, 4) if h <= Hkv]
    for hg in hgs:
        for pol in (pkv.Policy(tile_tokens=32, num_splits=1, kernel=kernel, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=5, kernel=kernel, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=16, num_splits=3, kernel=kernel, heads_per_cta=hg, merge_mode=pkv.MERGE_FUSED,
                               route=pkv.ROUTE_RECT),
                    pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, kernel=kernel,
                               heads_per_cta=hg)):
            _, _, ws = _check(dp, pol, ref, "G16 hg%d %s" % (hg, pol))
            tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
            want = wq.build_workqueue(RAGGED, Hkv, oracle_policy(pol))
            assert tasks.tolist() == [list(t) for t in want.tasks] and offs.tolist() == want.split_offsets
        if kernel == pkv.KERNEL_SIMT:
            break       # heads_per_cta only concerns the TMA kernel


def test_g16_many_units_and_partials():
    """G = 16 with more units than SMs and long units (ring wraps, dynamic hand-out at HG = 4), and the
    partial states of both head blocks against the oracle's split states through the merge."""
    rng = np.random.Generator(np.random.PCG64(17))
    lens = list(rng.integers(1, 3000, size=96))
    p = make_problem(lens, seed=711, Hq=64, Hkv=4)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(tile_tokens=32, num_splits=4), pkv.Policy(tile_tokens=32, num_splits=1),
                pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_FIXED_CHUNK, num_splits=0, chunk_tiles=8, merge_mode=pkv.MERGE_FUSED)):
        for hg in (4, 2, 1):
            pol.heads_per_cta = hg
            for _ in range(2):
                _check(dp, pol, ref, "hg%d %s" % (hg, pol))
    with pytest.raises(pkv.PkvError):
        dp.decode(pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=8))


@pytest.mark.parametrize("d", [64, 256])
@pytest.mark.parametrize("Hkv", [8, 4])
def test_head_dimensions_ragged_sweep(d, Hkv):
    """d = 64 and d = 256 on the TMA kernel, G = 4 and G = 8: every heads-per-CTA
    variant, both routes, separate / fused / channel-sliced merge, page size 32 as well."""
    for P in (16, 32):
        p = make_problem(RAGGED, seed=800 + d + Hkv + P, Hkv=Hkv, d=d, page_size=P)
        dp = DevProblem(p)
        ref = oracle_attention(p)
        for hg in (0, 1, 2, 4, 8):
            if hg > Hkv or (hg == 8 and d == 256):
                continue
            for pol in (pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=hg),
                        pkv.Policy(tile_tokens=32, num_splits=5, heads_per_cta=hg),
                        pkv.Policy(tile_tokens=32, num_splits=40, heads_per_cta=hg),          # sliced merge when B*Hq is small
                        pkv.Policy(tile_tokens=32, num_splits=3, heads_per_cta=hg, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT),
                        pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, heads_per_cta=hg)):
                _, _, ws = _check(dp, pol, ref, "d%d P%d hg%d %s" % (d, P, hg, pol))
        tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
        want = wq.build_workqueue(RAGGED, Hkv, oracle_policy(pol))
        assert tasks.tolist() == [list(t) for t in want.tasks]


@pytest.mark.parametrize("d", [64, 256])
@pytest.mark.parametrize("Hq,Hkv", [(32, 32), (32, 16), (64, 4), (32, 2)])
def test_head_dimensions_other_group_sizes(d, Hq, Hkv):
    """d = 64 and d = 256 with G = 1, 2 and 16: every heads-per-CTA variant (at most 4 with G = 16 or
    d = 256), both routes, separate / fused / channel-sliced merge."""
    G = Hq // Hkv
    p = make_problem(RAGGED, seed=860 + d + Hq + Hkv, Hq=Hq, Hkv=Hkv, d=d)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for hg in (0, 1, 2, 4, 8):
        if hg > Hkv or (hg == 8 and (d == 256 or G == 16)):
            continue
        for pol in (pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=5, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=40, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=3, heads_per_cta=hg, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT),
                    pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, heads_per_cta=hg)):
            _, _, ws = _check(dp, pol, ref, "d%d G%d Hkv%d hg%d %s" % (d, G, Hkv, hg, pol))
    tasks, offs = pkv.pkv_read_workqueue(dp.shape, pol, ws)
    want = wq.build_workqueue(RAGGED, Hkv, oracle_policy(pol))
    assert tasks.tolist() == [list(t) for t in want.tasks]


@pytest.mark.parametrize("d", [64, 256])
def test_head_dimensions_single_long_row_and_token_counts(d):
    """One long row (B = 1: the channel-sliced merge over 4 or 8 CTAs per head) and the K = 0
    counting pin at d = 64 / 256; d with the SIMT kernel is refused, not mis-computed."""
    p = make_problem([9000], seed=900 + d, d=d)
    dp = DevProblem(p)
    ref = oracle_attention(p)
    for pol in (pkv.Policy(tile_tokens=32, num_splits=64), pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0),
                pkv.Policy(tile_tokens=32, num_splits=16)):
        _check(dp, pol, ref, "d%d %s" % (d, pol))
    lens = [4097, 33, 1, 1000]
    p = make_problem(lens, seed=41 + d, d=d)
    p.k_cache[...] = 0
    p.v_cache[...] = np.random.Generator(np.random.PCG64(7)).integers(-8, 9, size=p.v_cache.shape).astype(np.float16)
    dp = DevProblem(p)
    pol = pkv.Policy(tile_tokens=32, num_splits=7)
    out, lse, ws = dp.decode(pol)
    assert_within_tolerance(out, oracle_attention(p)[0])
    q = wq.build_workqueue(lens, 8, oracle_policy(pol))
    m, l, a = read_partials(dp, pol, ws, q.num_tasks)
    for (row, kvh, split, tb, te) in q.tasks:
        n_i = q.split_offsets[row + 1] - q.split_offsets[row]
        if n_i > 1:
            slot = q.split_offsets[row] * 8 + kvh * n_i + split
            assert np.all(l[slot] == min(te * 32, lens[row]) - tb * 32) and np.all(m[slot] == 0.0)
    with pytest.raises(pkv.PkvError):
        dp.decode(pkv.Policy(tile_tokens=32, num_splits=2, kernel=pkv.KERNEL_SIMT))
