"""GPU parity for the fused KV-append (+RoPE) step ("fused
RoPE/KV-cache writes"; reading A29): pkv_decode_append against oracle/append_oracle.py --
outputs within tolerance, and the K/V bytes the kernel writes to the pool bit-exact."""
import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
from gpu_helpers import DevProblem, oracle_policy, to_dev
from helpers import assert_within_tolerance, make_problem
from oracle import append_oracle as ao

pytestmark = pytest.mark.gpu


def rope_tables(positions, d, base=10000.0):
    inv = base ** (-np.arange(0, d // 2, dtype=np.float64) * 2.0 / d)
    ang = np.arange(positions, dtype=np.float64)[:, None] * inv[None, :]
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)


def run_append(dp, p, pol, k_new, v_new, cos, sin, lens):
    dp.sl.copy_(to_dev(lens))
    ws = pkv.alloc_workspace(dp.shape, pol)
    dp.out.fill_(float("nan"))
    dp.lse.fill_(float("nan"))
    app = pkv.Append(k_new=to_dev(k_new), v_new=to_dev(v_new), rope_cos=None if cos is None else to_dev(cos),
                     rope_sin=None if sin is None else to_dev(sin), rope_positions=0 if cos is None else cos.shape[0])
    pkv.pkv_decode_append(dp.shape, pol, dp.q, dp.k, dp.v, dp.bt, dp.sl, None, app, dp.out, dp.lse, scale=p.scale, workspace=ws)
    torch.cuda.synchronize()
    return dp.out.cpu().numpy().astype(np.float64), dp.lse.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("Hkv", [8, 4, 16, 32, 2])          # G = 4, 8, 2, 1, 16
@pytest.mark.parametrize("rope", [True, False])
def test_append_step_matches_the_oracle_and_writes_the_pool_bit_exact(Hkv, rope):
    lens = np.array([1, 16, 17, 100, 0, 257, 700, 4099, 32, 33], dtype=np.int32)
    p = make_problem(list(lens), seed=1300 + Hkv)
    rng = np.random.Generator(np.random.PCG64(Hkv))
    p = make_problem(list(lens), seed=1300 + Hkv, Hkv=Hkv)
    k_new = rng.standard_normal((p.B, Hkv, 128)).astype(np.float16)
    v_new = rng.standard_normal((p.B, Hkv, 128)).astype(np.float16)
    cos, sin = rope_tables(4200, 128) if rope else (None, None)
    ref, ref_lse, k2, v2 = ao.append_and_attend(p.q, p.k_cache, p.v_cache, k_new, v_new, p.block_table, lens, cos, sin,
                                                 Hkv=Hkv, page_size=16, scale=p.scale)
    for pol in (pkv.Policy(tile_tokens=32, num_splits=1), pkv.Policy(tile_tokens=32, num_splits=5),
                pkv.Policy(tile_tokens=16, num_splits=3, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT, heads_per_cta=1),
                pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, heads_per_cta=2),
                pkv.Policy(tile_tokens=32, num_splits=4, heads_per_cta=min(4, Hkv))):
        dp = DevProblem(p)          # fresh pool: the step writes it
        out, lse = run_append(dp, p, pol, k_new, v_new, cos, sin, lens)
        assert not np.isnan(out).any()
        assert_within_tolerance(out, ref, "append Hkv%d rope%d %s" % (Hkv, rope, pol))
        fin = np.isfinite(ref_lse)
        assert np.array_equal(np.isneginf(lse), np.isneginf(ref_lse)) and np.abs(lse[fin] - ref_lse[fin]).max() <= 2e-3
        assert np.array_equal(dp.k.cpu().numpy().view(np.uint16), k2.view(np.uint16)), pol
        assert np.array_equal(dp.v.cpu().numpy().view(np.uint16), v2.view(np.uint16)), pol


def test_append_loop_grows_rows_across_pages_and_page_sizes():
    """Six consecutive fused steps (every row gains a token per step, crossing block and page
    boundaries) at page size 32: each step's output and the pool after the loop match the oracle
    applied step by step."""
    lens0 = np.array([30, 63, 14, 2000], dtype=np.int32)
    p = make_problem(list(lens0 + 8), seed=1400, page_size=32)
    dp = DevProblem(p)
    cos, sin = rope_tables(2100, 128)
    kc, vc = p.k_cache.copy(), p.v_cache.copy()
    rng = np.random.Generator(np.random.PCG64(2))
    pol = pkv.Policy(tile_tokens=32, num_splits=4)
    for t in range(1, 7):
        lens = (lens0 + t).astype(np.int32)
        k_new = rng.standard_normal((p.B, 8, 128)).astype(np.float16)
        v_new = rng.standard_normal((p.B, 8, 128)).astype(np.float16)
        ref, _, kc, vc = ao.append_and_attend(p.q, kc, vc, k_new, v_new, p.block_table, lens, cos, sin, Hkv=8, page_size=32,
                                               scale=p.scale)
        out, _ = run_append(dp, p, pol, k_new, v_new, cos, sin, lens)
        assert_within_tolerance(out, ref, "step %d" % t)
    assert np.array_equal(dp.k.cpu().numpy().view(np.uint16), kc.view(np.uint16))
    assert np.array_equal(dp.v.cpu().numpy().view(np.uint16), vc.view(np.uint16))


def test_append_unsupported_combinations_are_refused():
    p = make_problem([100], seed=5, d=64)                   # the append is compiled for d = 128
    dp = DevProblem(p)
    kn = np.zeros((1, 8, 64), np.float16)
    with pytest.raises(pkv.PkvError):
        run_append(dp, p, pkv.Policy(tile_tokens=32, num_splits=2), kn, kn, None, None, np.array([100], np.int32))
    p = make_problem([100], seed=6)
    dp = DevProblem(p)
    kn = np.zeros((1, 8, 128), np.float16)
    with pytest.raises(pkv.PkvError):
        run_append(dp, p, pkv.Policy(tile_tokens=32, num_splits=2, kernel=pkv.KERNEL_SIMT), kn, kn, None, None, np.array([100], np.int32))


# ------------------------------------------------------------------ one-byte caches (reading A30)

def run_append_q8(fp, pol, k_new, v_new, cos, sin, lens):
    """pkv_decode_append on the device state of a test_gpu_fp8.Fp8Problem (its pools are written)."""
    fp.sl.copy_(to_dev(lens))
    ws = pkv.alloc_workspace(fp.shape, pol)
    fp.out.fill_(float("nan"))
    fp.lse.fill_(float("nan"))
    app = pkv.Append(k_new=to_dev(k_new), v_new=to_dev(v_new), rope_cos=None if cos is None else to_dev(cos),
                     rope_sin=None if sin is None else to_dev(sin), rope_positions=0 if cos is None else cos.shape[0])
    pkv.pkv_decode_append(fp.shape, pol, fp.q, fp.k, fp.v, fp.bt, fp.sl, None, app, fp.out, fp.lse, scale=fp.p.scale, workspace=ws)
    torch.cuda.synchronize()
    return fp.out.cpu().numpy().astype(np.float64), fp.lse.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("kind", [pkv.KV_E4M3, pkv.KV_INT8])
@pytest.mark.parametrize("Hkv", [8, 4, 16, 32, 2])          # G = 4, 8, 2, 1, 16
@pytest.mark.parametrize("rope", [True, False])
def test_one_byte_append_step_matches_the_oracle_and_writes_the_pool_bit_exact(Hkv, rope, kind):
    """FP8 (E4M3) and INT8 caches, G = 4, 8, 2, 1, 16: the new token is quantised inside the decode launch
    (FP32 division by the head's scale, one rounding); outputs within tolerance, pool bytes bit-exact.
    Some elements of the new tokens saturate the code range."""
    from test_gpu_fp8 import Fp8Problem
    lens = np.array([1, 16, 17, 100, 0, 257, 700, 4099, 32, 33], dtype=np.int32)
    rng = np.random.Generator(np.random.PCG64(100 + Hkv))
    k_new = (3.0 * rng.standard_normal((len(lens), Hkv, 128))).astype(np.float16)   # K only moves scores: wide, INT8 clamps
    v_new = rng.standard_normal((len(lens), Hkv, 128)).astype(np.float16)           # outputs stay O(1): the tolerance is absolute
    k_new[2, 0, :4] = [60.0, -60.0, 1000.0, -65504.0]      # beyond 448 * scale (127 * scale): saturates, never NaN
    v_new[7, 0, :2] = [40.0, -40.0]                         # row of 4099 tokens: a saturated V with a small weight
    cos, sin = rope_tables(4200, 128) if rope else (None, None)
    for pol in (pkv.Policy(tile_tokens=32, num_splits=1), pkv.Policy(tile_tokens=32, num_splits=5),
                pkv.Policy(tile_tokens=16, num_splits=3, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT, heads_per_cta=1),
                pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, heads_per_cta=2),
                pkv.Policy(tile_tokens=32, num_splits=4, heads_per_cta=min(4, Hkv))):
        fp = Fp8Problem(list(lens), seed=1500 + Hkv, Hkv=Hkv, kind=kind)          # fresh pools: the step writes them
        ref, ref_lse, k2, v2 = ao.append_and_attend_q8(fp.p.q, fp.k8, fp.v8, fp.ks, fp.vs, k_new, v_new, fp.p.block_table, lens, cos, sin,
                                                        Hkv=Hkv, page_size=16, scale=fp.p.scale, kv_kind=2 if kind == pkv.KV_INT8 else 1)
        out, lse = run_append_q8(fp, pol, k_new, v_new, cos, sin, lens)
        what = "one-byte append kind%d Hkv%d rope%d %s" % (kind, Hkv, rope, pol)
        assert not np.isnan(out).any(), what
        assert_within_tolerance(out, ref, what)
        fin = np.isfinite(ref_lse)
        assert np.array_equal(np.isneginf(lse), np.isneginf(ref_lse)) and np.abs(lse[fin] - ref_lse[fin]).max() <= 2e-3, what
        assert np.array_equal(fp.k.cpu().numpy(), k2), what
        assert np.array_equal(fp.v.cpu().numpy(), v2), what


@pytest.mark.parametrize("kind", [pkv.KV_E4M3, pkv.KV_INT8])
def test_one_byte_append_loop_grows_rows_across_pages(kind):
    """Six consecutive fused steps on one-byte caches at page size 32 (NULL scales on the INT8 run =
    scale 1): each step's output and the pools after the loop match the oracle applied step by step."""
    from test_gpu_fp8 import Fp8Problem
    lens0 = np.array([30, 63, 14, 2000], dtype=np.int32)
    fp = Fp8Problem(list(lens0 + 8), seed=1600, page_size=32, kind=kind, scales=kind == pkv.KV_E4M3)
    cos, sin = rope_tables(2100, 128)
    kc, vc = fp.k8.copy(), fp.v8.copy()
    rng = np.random.Generator(np.random.PCG64(4))
    pol = pkv.Policy(tile_tokens=32, num_splits=4)
    for t in range(1, 7):
        lens = (lens0 + t).astype(np.int32)
        k_new = rng.standard_normal((4, 8, 128)).astype(np.float16)
        v_new = rng.standard_normal((4, 8, 128)).astype(np.float16)
        ref, _, kc, vc = ao.append_and_attend_q8(fp.p.q, kc, vc, fp.ks, fp.vs, k_new, v_new, fp.p.block_table, lens, cos, sin,
                                                  Hkv=8, page_size=32, scale=fp.p.scale, kv_kind=2 if kind == pkv.KV_INT8 else 1)
        out, _ = run_append_q8(fp, pol, k_new, v_new, cos, sin, lens)
        assert_within_tolerance(out, ref, "kind %d step %d" % (kind, t))
    assert np.array_equal(fp.k.cpu().numpy(), kc) and np.array_equal(fp.v.cpu().numpy(), vc)
