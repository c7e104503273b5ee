"""Pins for the FP64 attention oracle (oracle/pkv_oracle.c): nothing here comes from the CUDA path.

P1 brute-force dense numpy (Eq. 1)          P4 split-count invariance
P2 page-pool permutation invariance  P5 dominant key at every boundary
P3 K = 0  =>  O = mean(V), exact with integer V         P6 N = 1, N = 2, equal-keys closed forms
"""
import math

import numpy as np
import pytest

from helpers import (Problem, default_scale, dense_attention_bruteforce, make_problem, permute_pool,
                     token_location)
from oracle import pkv_oracle, workqueue_oracle as wq
from pkv_inputs import PAD_PAGE


def oracle_attention(p: Problem, **kw):
    return pkv_oracle.attention(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens, Hkv=p.Hkv,
                                page_size=p.page_size, scale=p.scale, **kw)


def test_half_decoder_all_bit_patterns():
    """The oracle's own FP16 decoder against numpy's float16 on all 65536 patterns."""
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float64)
    for b in range(65536):
        got = pkv_oracle.half_to_double(b)
        if math.isnan(ref[b]):
            assert math.isnan(got)
        else:
            assert got == ref[b] and math.copysign(1.0, got) == math.copysign(1.0, ref[b]), b


@pytest.mark.parametrize("Hkv", [8, 4])
@pytest.mark.parametrize("lens", [[1], [2], [15, 16, 17], [31, 32, 33], [100, 1, 40]])
def test_p1_bruteforce_dense(lens, Hkv):
    p = make_problem(lens, seed=11 + len(lens) + Hkv, Hkv=Hkv)
    out, lse = oracle_attention(p)
    ref, ref_lse = dense_attention_bruteforce(p)
    assert np.abs(out - ref).max() <= 1e-12
    assert np.abs(lse - ref_lse).max() <= 1e-12


def test_p1_bruteforce_other_shapes():
    """A transposed operand or a wrong head map shows up when Hq, Hkv, d and P all differ."""
    p = make_problem([37, 5], seed=5, Hq=6, Hkv=3, d=24, page_size=4)
    out, lse = oracle_attention(p)
    ref, ref_lse = dense_attention_bruteforce(p)
    assert np.abs(out - ref).max() <= 1e-12
    assert np.abs(lse - ref_lse).max() <= 1e-12


def test_p2_page_pool_permutation_invariance_bit_identical():
    p = make_problem([100, 33, 16], seed=21)
    out, lse = oracle_attention(p)
    p2 = permute_pool(p, seed=99)
    assert not np.array_equal(p.block_table, p2.block_table)
    out2, lse2 = oracle_attention(p2)
    assert np.array_equal(out, out2) and np.array_equal(lse, lse2)


def test_strided_layout_reading_a1():
    """The paper's [page, Hkv, page_size, d] layout through explicit strides gives the
    same bits as the BASELINE.json layout [page, page_size, Hkv, d]."""
    p = make_problem([70, 19], seed=31)
    out, lse = oracle_attention(p)
    k_hnd = np.ascontiguousarray(p.k_cache.transpose(0, 2, 1, 3))
    v_hnd = np.ascontiguousarray(p.v_cache.transpose(0, 2, 1, 3))
    P, H, d = p.page_size, p.Hkv, p.d
    out2, lse2 = pkv_oracle.attention(p.q, k_hnd, v_hnd, p.block_table, p.seq_lens, Hkv=H, page_size=P,
                                      scale=p.scale, strides=(H * P * d, d, P * d))
    assert np.array_equal(out, out2) and np.array_equal(lse, lse2)


def test_p3_zero_keys_give_mean_of_values_exactly():
    p = make_problem([100, 47], seed=41)
    rng = np.random.Generator(np.random.PCG64(7))
    p.k_cache[...] = 0
    p.v_cache[...] = rng.integers(-8, 9, size=p.v_cache.shape).astype(np.float16)
    out, lse = oracle_attention(p)
    for i in range(p.B):
        N = int(p.seq_lens[i])
        for g in range(p.Hkv):
            acc = np.zeros(p.d)
            for j in range(N):
                page, r = token_location(p, i, j)
                acc += p.v_cache[page, r, g].astype(np.float64)
            mean = acc / N                      # small integers: the sum is exact
            for hh in range(p.G):
                assert np.abs(out[i, g * p.G + hh] - mean).max() <= 1e-15
                assert abs(lse[i, g * p.G + hh] - math.log(N)) <= 1e-14


def test_a10_tail_and_unused_entries_never_read():
    """Tokens >= N_i in the last page hold huge values and NaN, the unused block-table entries
    hold PAD_PAGE; the result must not move (reading A10)."""
    p = make_problem([37, 50], seed=51, reserve_extra=40)
    out, lse = oracle_attention(p)
    k2, v2 = p.k_cache.copy(), p.v_cache.copy()
    owned = set()
    for i in range(p.B):
        for j in range(int(p.seq_lens[i])):
            owned.add(token_location(p, i, j))
    for page in range(k2.shape[0]):
        for r in range(p.page_size):
            if (page, r) not in owned:
                k2[page, r] = np.float16(60000.0)
                v2[page, r] = np.float16(np.nan)
    t2 = p.block_table.copy()
    for i in range(p.B):
        t2[i, math.ceil(int(p.seq_lens[i]) / p.page_size):] = PAD_PAGE
    out2, lse2 = pkv_oracle.attention(p.q, k2, v2, t2, p.seq_lens, Hkv=p.Hkv, page_size=p.page_size,
                                      scale=p.scale)
    assert np.array_equal(out, out2) and np.array_equal(lse, lse2)


@pytest.mark.parametrize("S", [1, 2, 3, 4, 16, 64, 200])
def test_p4_split_count_invariance(S):
    """Split states merged by PAPER.md:60-61 equal Eq. (1) for any split count,
    including S > T where trailing splits are empty."""
    p = make_problem([1000, 95, 32, 1], seed=61)
    ref, ref_lse = oracle_attention(p)
    pol = wq.Policy(tile_tokens=32, num_splits=S)
    q = wq.build_workqueue(p.seq_lens, p.Hkv, pol)
    out, lse = pkv_oracle.attention_via_splits(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens,
                                               np.array(q.tasks, dtype=np.int32), q.split_offsets,
                                               Hkv=p.Hkv, page_size=p.page_size, tile_tokens=32,
                                               scale=p.scale)
    assert np.abs(out - ref).max() <= 1e-12
    assert np.abs(lse - ref_lse).max() <= 1e-12


def test_p4_rect_route_neutral_states():
    """Rectangular grid: empty splits carry (m, l, a) = (-inf, 0, 0) and drop out."""
    p = make_problem([40, 700, 0], seed=62)
    ref, ref_lse = oracle_attention(p)
    pol = wq.Policy(tile_tokens=32, num_splits=8, route=wq.ROUTE_RECT)
    q = wq.build_workqueue(p.seq_lens, p.Hkv, pol)
    tasks = np.array(q.tasks, dtype=np.int32)
    m, l, a = pkv_oracle.split_states(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens, tasks,
                                      Hkv=p.Hkv, page_size=p.page_size, tile_tokens=32, scale=p.scale)
    empty = tasks[:, 3] >= tasks[:, 4]
    assert empty.sum() == q.empty_ctas > 0
    assert np.all(np.isneginf(m[empty])) and np.all(l[empty] == 0) and np.all(a[empty] == 0)
    out, lse = pkv_oracle.attention_via_splits(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens,
                                               tasks, q.split_offsets, Hkv=p.Hkv,
                                               page_size=p.page_size, tile_tokens=32, scale=p.scale)
    assert np.abs(out - ref).max() <= 1e-12
    assert np.all(out[2] == 0) and np.all(np.isneginf(lse[2]))          # reading A9


def test_merge_associative_and_neutral():
    rng = np.random.Generator(np.random.PCG64(3))
    n, d = 7, 16
    m = rng.standard_normal(n) * 5
    l = rng.random(n) + 0.5
    a = rng.standard_normal((n, d))
    o_all, lse_all = pkv_oracle.merge(m, l, a)
    # closed form of the definition: O = sum_s e^{m_s} a_s / sum_s e^{m_s} l_s
    w = np.exp(m - m.max())
    assert np.abs(o_all - (w[:, None] * a).sum(0) / (w * l).sum()).max() <= 1e-13
    assert abs(lse_all - (m.max() + math.log((w * l).sum()))) <= 1e-13
    # adding neutral states changes nothing
    m2 = np.concatenate([m, [-np.inf, -np.inf]])
    l2 = np.concatenate([l, [0.0, 0.0]])
    a2 = np.concatenate([a, np.zeros((2, d))])
    o2, lse2 = pkv_oracle.merge(m2, l2, a2)
    assert np.array_equal(o2, o_all) and lse2 == lse_all
    # all neutral -> O = 0, LSE = -inf (reading A9)
    o3, lse3 = pkv_oracle.merge(np.full(3, -np.inf), np.zeros(3), np.zeros((3, d)))
    assert np.all(o3 == 0) and lse3 == -np.inf


def _dominant_positions(N, page_size, tile, splits):
    pos = {0, N - 1}
    for unit in (page_size, tile):
        for b in range(unit, N, unit):
            pos.update({b - 1, b, b + 1})
    T = math.ceil(N / tile)
    c = math.ceil(T / splits)
    for s in range(1, splits):
        b = s * c * tile
        pos.update({b - 1, b, b + 1})
    return sorted(x for x in pos if 0 <= x < N)


def test_p5_dominant_key_selects_that_value():
    """k_{j*} = 3 q for all G heads sharing one q  =>  x* >> the rest  =>  O = v_{j*}."""
    N = 200
    base = make_problem([N], seed=71)
    for hh in range(1, base.G):                 # one q per KV group so a single key dominates all G heads
        base.q[0, hh::base.G] = base.q[0, 0::base.G]
    positions = _dominant_positions(N, base.page_size, 32, 4)
    assert len(positions) > 30
    for jstar in positions:
        k2 = base.k_cache.copy()
        page, r = token_location(base, 0, jstar)
        for g in range(base.Hkv):
            k2[page, r, g] = (3.0 * base.q[0, g * base.G].astype(np.float32)).astype(np.float16)
        out, _ = pkv_oracle.attention(base.q, k2, base.v_cache, base.block_table, base.seq_lens,
                                      Hkv=base.Hkv, page_size=base.page_size, scale=base.scale)
        for h in range(base.Hq):
            want = base.v_cache[page, r, h // base.G].astype(np.float64)
            assert np.abs(out[0, h] - want).max() < 1e-6, (jstar, h)


def test_p6_closed_forms_n1_n2_equal_keys():
    # N = 1: O = v_0 exactly, LSE = x_0
    p = make_problem([1], seed=81)
    out, lse = oracle_attention(p)
    page, r = token_location(p, 0, 0)
    for h in range(p.Hq):
        g = h // p.G
        assert np.array_equal(out[0, h], p.v_cache[page, r, g].astype(np.float64))
        x0 = p.scale * float(p.q[0, h].astype(np.float64) @ p.k_cache[page, r, g].astype(np.float64))
        assert abs(lse[0, h] - x0) <= 1e-13
    # N = 2: O = sigma(x0 - x1) v0 + sigma(x1 - x0) v1
    p = make_problem([2], seed=82)
    out, _ = oracle_attention(p)
    (p0, r0), (p1, r1) = token_location(p, 0, 0), token_location(p, 0, 1)
    for h in range(p.Hq):
        g = h // p.G
        qv = p.q[0, h].astype(np.float64)
        x0 = p.scale * float(qv @ p.k_cache[p0, r0, g].astype(np.float64))
        x1 = p.scale * float(qv @ p.k_cache[p1, r1, g].astype(np.float64))
        s0 = 1.0 / (1.0 + math.exp(x1 - x0))
        want = s0 * p.v_cache[p0, r0, g].astype(np.float64) + (1 - s0) * p.v_cache[p1, r1, g].astype(np.float64)
        assert np.abs(out[0, h] - want).max() <= 1e-13
    # all keys equal: uniform weights, O = mean(V) (V integer => exact sum)
    p = make_problem([53], seed=83)
    rng = np.random.Generator(np.random.PCG64(1))
    p.k_cache[...] = p.k_cache[0, 0, 0][None, None, None, :]
    p.v_cache[...] = rng.integers(-4, 5, size=p.v_cache.shape).astype(np.float16)
    out, _ = oracle_attention(p)
    for g in range(p.Hkv):
        acc = np.zeros(p.d)
        for j in range(53):
            page, r = token_location(p, 0, j)
            acc += p.v_cache[page, r, g].astype(np.float64)
        for hh in range(p.G):
            assert np.abs(out[0, g * p.G + hh] - acc / 53).max() <= 1e-13


def test_scale_is_applied_to_scores():
    """Doubling the scale is the same as doubling q (exact in FP16: power of two)."""
    p = make_problem([60], seed=91)
    p.q[...] = (p.q.astype(np.float32) * 0.25).astype(np.float16)
    out_a, lse_a = pkv_oracle.attention(p.q, p.k_cache, p.v_cache, p.block_table, p.seq_lens, Hkv=p.Hkv,
                                        page_size=p.page_size, scale=2.0 * p.scale)
    q2 = (p.q.astype(np.float32) * 2).astype(np.float16)
    out_b, lse_b = pkv_oracle.attention(q2, p.k_cache, p.v_cache, p.block_table, p.seq_lens, Hkv=p.Hkv,
                                        page_size=p.page_size, scale=p.scale)
    assert np.abs(out_a - out_b).max() <= 1e-13 and np.abs(lse_a - lse_b).max() <= 1e-12
    assert default_scale(128) == float(np.float32(1 / math.sqrt(128)))


# ---------------------------------------------------------------- FP8 (E4M3) KV, reading A28

def test_e4m3_decoder_all_bit_patterns_and_closed_forms():
    """The oracle's own E4M3 decoder on all 256 codes against torch.float8_e4m3fn (a library
    routine), and against what the format fixes: 1.0 = 0x38, largest finite 448 = 0x7E, smallest
    subnormal 2^-9, smallest normal 2^-6, one NaN code per sign, no infinity, monotone codes."""
    import torch
    want = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    got = np.array([pkv_oracle.e4m3_to_double(b) for b in range(256)])
    assert np.array_equal(np.isnan(got), np.isnan(want))
    ok = ~np.isnan(want)
    assert np.array_equal(got[ok], want[ok]) and np.array_equal(np.signbit(got[ok]), np.signbit(want[ok]))
    assert got[0x38] == 1.0 and got[0x7E] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6
    assert np.isnan(got[0x7F]) and np.isnan(got[0xFF]) and not np.isinf(got).any()
    assert np.all(np.diff(got[:0x7F]) > 0) and np.array_equal(got[0x80:0xFF], -got[:0x7F])


def _quantize_e4m3(x: np.ndarray, scale: np.ndarray):
    """x [pages, P, Hkv, d] / scale[g] rounded to E4M3 by torch (bytes), per KV head."""
    import torch
    t = torch.from_numpy((x.astype(np.float32) / scale[None, None, :, None].astype(np.float32)))
    return t.to(torch.float8_e4m3fn).view(torch.uint8).numpy().copy()


def test_fp8_attention_reduces_to_the_fp16_oracle_and_to_brute_force():
    """With power-of-two scales every dequantised value scale * e4m3 is exactly an FP16 number, so
    the FP8 entry point must agree with the (pinned) FP16 entry point on the dequantised caches to
    rounding order; with arbitrary scales it must agree with dense numpy on the real values.  A
    swapped K/V scale, a scale indexed by the wrong head or a mis-decoded byte fails one of them."""
    p = make_problem([1, 17, 100, 0, 33], seed=61)
    ks = np.array([0.5, 1.0, 2.0, 0.25, 4.0, 0.125, 1.0, 8.0])
    vs = np.array([2.0, 0.5, 1.0, 4.0, 0.25, 1.0, 0.125, 0.5])
    k8, v8 = _quantize_e4m3(p.k_cache, ks), _quantize_e4m3(p.v_cache, vs)
    dec = np.vectorize(pkv_oracle.e4m3_to_double)
    kd = (dec(k8) * ks[None, None, :, None]).astype(np.float16)
    vd = (dec(v8) * vs[None, None, :, None]).astype(np.float16)
    assert np.array_equal(kd.astype(np.float64), dec(k8) * ks[None, None, :, None])      # exact in FP16
    got, got_lse = pkv_oracle.attention_fp8(p.q, k8, v8, ks, vs, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    ref, ref_lse = pkv_oracle.attention(p.q, kd, vd, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    assert np.abs(got - ref).max() <= 1e-12
    fin = np.isfinite(ref_lse)
    assert np.array_equal(np.isneginf(got_lse), np.isneginf(ref_lse)) and np.abs(got_lse[fin] - ref_lse[fin]).max() <= 1e-12
    # arbitrary scales: dense numpy on the real values
    ks2, vs2 = np.linspace(0.03, 0.11, 8), np.linspace(0.9, 0.05, 8)
    got, got_lse = pkv_oracle.attention_fp8(p.q, k8, v8, ks2, vs2, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    pr = Problem(q=p.q, k_cache=dec(k8) * ks2[None, None, :, None], v_cache=dec(v8) * vs2[None, None, :, None],
                 block_table=p.block_table, seq_lens=p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    ref, ref_lse = dense_attention_bruteforce(pr)
    assert np.abs(got - ref).max() <= 1e-12 and np.abs(got_lse[fin] - ref_lse[fin]).max() <= 1e-12
    # swapping the scales changes the result (the test can see them)
    bad, _ = pkv_oracle.attention_fp8(p.q, k8, v8, vs2, ks2, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    assert np.abs(bad - ref).max() > 1e-3


# ---------------------------------------------------------------- fused KV-append + RoPE, reading A29

def _rope_tables(positions, d, base=10000.0):
    inv = base ** (-np.arange(0, d // 2, dtype=np.float64) * 2.0 / d)
    ang = np.arange(positions, dtype=np.float64)[:, None] * inv[None, :]
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)


def test_rope_rotation_against_complex_multiplication_and_invariants():
    """The rotate-half formula restated as a complex product (x[c] + i x[c+d/2]) * e^{i theta}; pair
    norms are preserved; position 0 is the identity; scores depend on the position difference only."""
    from oracle import append_oracle as ao
    rng = np.random.Generator(np.random.PCG64(3))
    d = 128
    cos, sin = _rope_tables(5000, d)
    x = rng.standard_normal((7, d)).astype(np.float16)
    for pos in (0, 1, 17, 4999):
        y = ao.rope_rotate_f16(x, cos[pos], sin[pos]).astype(np.float64)
        z = (x[:, :64].astype(np.float64) + 1j * x[:, 64:].astype(np.float64)) * (cos[pos].astype(np.float64) + 1j * sin[pos].astype(np.float64))
        want = np.concatenate([z.real, z.imag], axis=-1)
        assert np.abs(y - want).max() <= 4e-3          # FP16 rounding of values up to ~4
        n_in = x[:, :64].astype(np.float64) ** 2 + x[:, 64:].astype(np.float64) ** 2
        assert np.abs((y[:, :64] ** 2 + y[:, 64:] ** 2) - n_in).max() <= 3e-2
    assert np.array_equal(ao.rope_rotate_f16(x, cos[0], sin[0]), x)
    # relative position: <R(q, m), R(k, n)> = <R(q, m + s), R(k, n + s)>
    q, k = x[0:1], x[1:2]
    a = (ao.rope_rotate_f16(q, cos[40], sin[40]).astype(np.float64) * ao.rope_rotate_f16(k, cos[25], sin[25]).astype(np.float64)).sum()
    b = (ao.rope_rotate_f16(q, cos[1040], sin[1040]).astype(np.float64) * ao.rope_rotate_f16(k, cos[1025], sin[1025]).astype(np.float64)).sum()
    assert abs(a - b) <= 5e-2


def test_append_step_against_dense_brute_force():
    """The fused step against numpy on a dense gathered copy: old tokens from the cache, the new
    token from (RoPE'd) k_new / v_new, q RoPE'd -- no cache-update code involved.  Also: only the slots
    of the new tokens change, rows with N = 0 change nothing, no tables = plain append."""
    from oracle import append_oracle as ao
    lens = np.array([1, 17, 100, 0, 33, 64], dtype=np.int32)
    p = make_problem(list(lens), seed=71)
    rng = np.random.Generator(np.random.PCG64(5))
    k_new = rng.standard_normal((p.B, 8, 128)).astype(np.float16)
    v_new = rng.standard_normal((p.B, 8, 128)).astype(np.float16)
    cos, sin = _rope_tables(256, 128)
    for tables in ((cos, sin), (None, None)):
        out, lse, k2, v2 = ao.append_and_attend(p.q, p.k_cache, p.v_cache, k_new, v_new, p.block_table, lens, tables[0], tables[1],
                                                 Hkv=8, page_size=16, scale=p.scale)
        changed = np.zeros(p.k_cache.shape[:2], dtype=bool)
        for i in range(p.B):
            N = int(lens[i])
            if N == 0:
                assert np.all(out[i] == 0) and np.all(np.isneginf(lse[i]))
                continue
            pos = N - 1
            kn = ao.rope_rotate_f16(k_new[i], cos[pos], sin[pos]) if tables[0] is not None else k_new[i]
            qn = ao.rope_rotate_f16(p.q[i], cos[pos], sin[pos]) if tables[0] is not None else p.q[i]
            Kd = np.stack([p.k_cache[p.block_table[i, j // 16], j % 16] for j in range(N - 1)] + [kn]).astype(np.float64)
            Vd = np.stack([p.v_cache[p.block_table[i, j // 16], j % 16] for j in range(N - 1)] + [v_new[i]]).astype(np.float64)
            for h in range(32):
                x = (Kd[:, h // 4, :] @ qn[h].astype(np.float64)) * p.scale
                w = np.exp(x - x.max())
                assert np.abs(out[i, h] - (w[:, None] * Vd[:, h // 4, :]).sum(0) / w.sum()).max() <= 1e-12
            changed[p.block_table[i, pos // 16], pos % 16] = True
            assert np.array_equal(k2[p.block_table[i, pos // 16], pos % 16], kn)
            assert np.array_equal(v2[p.block_table[i, pos // 16], pos % 16], v_new[i])
        assert np.array_equal(k2[~changed], p.k_cache[~changed]) and np.array_equal(v2[~changed], p.v_cache[~changed])


def test_int8_attention_reduces_to_the_fp16_oracle_and_to_brute_force():
    """INT8 caches (reading A28): with power-of-two scales every dequantised value is an FP16 number,
    so the INT8 entry point must agree with the FP16 oracle on the dequantised caches; with arbitrary
    scales with dense numpy on the real values (the byte decode here is numpy's own int8 view)."""
    p = make_problem([1, 17, 100, 0, 33], seed=63)
    rng = np.random.Generator(np.random.PCG64(9))
    k8 = rng.integers(-128, 128, size=p.k_cache.shape).astype(np.int8).view(np.uint8)
    v8 = rng.integers(-128, 128, size=p.v_cache.shape).astype(np.int8).view(np.uint8)
    ks = np.array([2.0 ** -5, 2.0 ** -6, 2.0 ** -4, 2.0 ** -7, 2.0 ** -5, 2.0 ** -6, 2.0 ** -5, 2.0 ** -8])
    vs = np.array([2.0 ** -6, 2.0 ** -5, 2.0 ** -7, 2.0 ** -4, 2.0 ** -6, 2.0 ** -5, 2.0 ** -6, 2.0 ** -5])
    kd = (k8.view(np.int8).astype(np.float64) * ks[None, None, :, None])
    vd = (v8.view(np.int8).astype(np.float64) * vs[None, None, :, None])
    assert np.array_equal(kd.astype(np.float16).astype(np.float64), kd)
    got, got_lse = pkv_oracle.attention_int8(p.q, k8, v8, ks, vs, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    ref, ref_lse = pkv_oracle.attention(p.q, kd.astype(np.float16), vd.astype(np.float16), p.block_table, p.seq_lens, Hkv=8,
                                        page_size=16, scale=p.scale)
    fin = np.isfinite(ref_lse)
    assert np.abs(got - ref).max() <= 1e-12 and np.abs(got_lse[fin] - ref_lse[fin]).max() <= 1e-12
    ks2, vs2 = np.linspace(0.003, 0.011, 8), np.linspace(0.02, 0.005, 8)
    got, got_lse = pkv_oracle.attention_int8(p.q, k8, v8, ks2, vs2, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    pr = Problem(q=p.q, k_cache=k8.view(np.int8).astype(np.float64) * ks2[None, None, :, None],
                 v_cache=v8.view(np.int8).astype(np.float64) * vs2[None, None, :, None],
                 block_table=p.block_table, seq_lens=p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    ref, ref_lse = dense_attention_bruteforce(pr)
    assert np.abs(got - ref).max() <= 1e-12 and np.abs(got_lse[fin] - ref_lse[fin]).max() <= 1e-12
    e4, _ = pkv_oracle.attention_fp8(p.q, k8, v8, ks2, vs2, p.block_table, p.seq_lens, Hkv=8, page_size=16, scale=p.scale)
    assert not np.allclose(np.nan_to_num(e4), got)          # the byte kind matters


def test_one_byte_quantisers_closed_forms_round_trip_and_torch():
    """Reading A30: FP32 -> E4M3 (nearest, ties to the even code, saturating at 448) and FP32 -> INT8
    (half to even, clamp to +-127).  Pinned by: every finite code survives decode -> encode (the decoder
    is pinned on all 256 codes above); ties / saturation / subnormals worked out by hand; sign symmetry
    and monotonicity; torch.float8_e4m3fn on the whole FP16 grid inside +-448."""
    import torch
    from oracle import append_oracle as ao
    codes = np.arange(0x7F, dtype=np.uint8)
    vals = np.array([pkv_oracle.e4m3_to_double(int(c)) for c in codes], dtype=np.float32)
    assert np.array_equal(ao.quantize_e4m3(vals), codes)
    assert np.array_equal(ao.quantize_e4m3(-vals[1:]), codes[1:] | 0x80)
    hand = {1.0: 0x38, 1.0625: 0x38, 1.1875: 0x3A, 1.0626: 0x39, 448.0: 0x7E, 464.0: 0x7E, 1000.0: 0x7E, 3e38: 0x7E,
            2.0 ** -9: 0x01, 2.0 ** -10: 0x00, 3 * 2.0 ** -11: 0x01, 3 * 2.0 ** -10: 0x02, 2.0 ** -6: 0x08, 0.0: 0x00,
            240.0: 0x77, 232.0: 0x76, 248.0: 0x78}      # 232 = tie 224|240 -> even code 0x76; 248 = tie 240|256 -> 0x78
    for x, c in hand.items():
        assert int(ao.quantize_e4m3(np.float32(x))) == c, (x, hex(c))
        if x > 0:
            assert int(ao.quantize_e4m3(np.float32(-x))) == c | 0x80
    assert int(ao.quantize_e4m3(np.float32("nan"))) == 0x7F and int(ao.quantize_e4m3(np.float32(-0.0))) == 0x80
    xs = np.sort(np.random.Generator(np.random.PCG64(3)).uniform(-500, 500, 20000).astype(np.float32))
    dec = np.array([pkv_oracle.e4m3_to_double(int(c)) for c in ao.quantize_e4m3(xs)])
    assert np.all(np.diff(dec) >= 0)                                        # monotone
    inside = np.abs(xs) <= 448
    assert np.all(np.abs(dec[inside] - xs[inside]) <= np.maximum(np.abs(xs[inside]) * 2.0 ** -4, 2.0 ** -10))   # half an ulp
    g = np.arange(65536, dtype=np.uint16).view(np.float16)
    g = g[np.isfinite(g) & (np.abs(g.astype(np.float32)) <= 448)].astype(np.float32)
    t = torch.from_numpy(g).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(ao.quantize_e4m3(g), t)
    i8 = ao.quantize_int8(np.array([0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 126.5, 127.4, 127.5, 300.0, -127.5, -128.0, -1e9, 0.49999997],
                                   dtype=np.float32)).view(np.int8)
    assert i8.tolist() == [0, 2, 2, 0, -2, -2, 126, 127, 127, 127, -127, -127, -127, 0]
    # the division is FP32: one correctly rounded quotient, then one rounding to the code
    tok = np.array([[3.0, 1.0, -7.0, 0.1]], dtype=np.float16)
    sc = np.array([0.3], dtype=np.float32)
    y = np.float32(tok.astype(np.float32)) / sc[0]
    assert np.array_equal(ao.quantize_token(tok, sc, 1), ao.quantize_e4m3(y)) and np.array_equal(ao.quantize_token(tok, sc, 2), ao.quantize_int8(y))


@pytest.mark.parametrize("kind", [1, 2])
def test_one_byte_append_step_against_dense_brute_force(kind):
    """Reading A30 against numpy on a dense gathered copy: old tokens dequantised from the cache bytes,
    the new token = scale * dec(code) with the code worked out here from numpy's own rounding of the
    FP32 quotient (INT8) or the nearest-table-value search (E4M3, cross-checked with torch), q RoPE'd.
    Only the new tokens' slots change; rows with N = 0 change nothing."""
    import torch
    from oracle import append_oracle as ao
    lens = np.array([1, 17, 100, 0, 33, 64], dtype=np.int32)
    p = make_problem(list(lens), seed=73)
    rng = np.random.Generator(np.random.PCG64(6))
    ks, vs = rng.uniform(0.03, 0.07, 8).astype(np.float32), rng.uniform(0.03, 0.07, 8).astype(np.float32)

    def to_codes(x32):
        if kind == 2:
            return np.clip(np.rint(x32), -127, 127).astype(np.int8).view(np.uint8)
        return torch.from_numpy(np.clip(x32, -448, 448).astype(np.float32)).to(torch.float8_e4m3fn).view(torch.uint8).numpy()

    def dec(codes):
        if kind == 2:
            return codes.view(np.int8).astype(np.float64)
        return torch.from_numpy(codes.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()

    k8 = to_codes(p.k_cache.astype(np.float32) / ks[None, None, :, None])
    v8 = to_codes(p.v_cache.astype(np.float32) / vs[None, None, :, None])
    k_new = rng.standard_normal((p.B, 8, 128)).astype(np.float16)
    v_new = rng.standard_normal((p.B, 8, 128)).astype(np.float16)
    cos, sin = _rope_tables(256, 128)
    for tables in ((cos, sin), (None, None)):
        out, lse, k2, v2 = ao.append_and_attend_q8(p.q, k8, v8, ks, vs, k_new, v_new, p.block_table, lens, tables[0], tables[1],
                                                    Hkv=8, page_size=16, scale=p.scale, kv_kind=kind)
        changed = np.zeros(k8.shape[:2], dtype=bool)
        for i in range(p.B):
            N = int(lens[i])
            if N == 0:
                assert np.all(out[i] == 0) and np.all(np.isneginf(lse[i]))
                continue
            pos = N - 1
            kn = ao.rope_rotate_f16(k_new[i], cos[pos], sin[pos]) if tables[0] is not None else k_new[i]
            qn = ao.rope_rotate_f16(p.q[i], cos[pos], sin[pos]) if tables[0] is not None else p.q[i]
            kc = to_codes((kn.astype(np.float32) / ks[:, None]).astype(np.float32))
            vc = to_codes((v_new[i].astype(np.float32) / vs[:, None]).astype(np.float32))
            page, slot = p.block_table[i, pos // 16], pos % 16
            assert np.array_equal(k2[page, slot], kc) and np.array_equal(v2[page, slot], vc)
            changed[page, slot] = True
            Kd = np.stack([dec(k8[p.block_table[i, j // 16], j % 16]) for j in range(N - 1)] + [dec(kc)]) * ks.astype(np.float64)[None, :, None]
            Vd = np.stack([dec(v8[p.block_table[i, j // 16], j % 16]) for j in range(N - 1)] + [dec(vc)]) * vs.astype(np.float64)[None, :, None]
            for h in range(32):
                x = (Kd[:, h // 4, :] @ qn[h].astype(np.float64)) * p.scale
                w = np.exp(x - x.max())
                assert np.abs(out[i, h] - (w[:, None] * Vd[:, h // 4, :]).sum(0) / w.sum()).max() <= 1e-12
        assert np.array_equal(k2[~changed], k8[~changed]) and np.array_equal(v2[~changed], v8[~changed])
