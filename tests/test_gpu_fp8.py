"""GPU parity for FP8 (E4M3) KV caches with in-loop dequantisation (
PAPER.md:271 "dequantization-aware paged decode"; reading A28).  Both sides see the
same bytes and the same per-KV-head scales; the oracle decodes E4M3 itself (pinned on all 256
codes, tests/test_oracle_pins.py)."""
import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
from gpu_helpers import oracle_policy, to_dev
from helpers import assert_within_tolerance, make_problem
from oracle import pkv_oracle, workqueue_oracle as wq

pytestmark = pytest.mark.gpu

RAGGED = [1, 2, 15, 16, 17, 31, 32, 33, 100, 0, 257, 700, 4099]


def quantize(x: np.ndarray, scale: np.ndarray, kind: int = 1) -> np.ndarray:
    y = x.astype(np.float32) / scale[None, None, :, None].astype(np.float32)
    if kind == pkv.KV_INT8:
        return np.clip(np.rint(y), -127, 127).astype(np.int8).view(np.uint8).copy()
    t = torch.from_numpy(np.clip(y, -448.0, 448.0))
    return t.to(torch.float8_e4m3fn).view(torch.uint8).numpy().copy()


class Fp8Problem:
    def __init__(self, lens, seed, Hkv=8, page_size=16, scales=True, kind=pkv.KV_E4M3, Hq=32):
        self.p = p = make_problem(lens, seed=seed, Hq=Hq, Hkv=Hkv, page_size=page_size)
        self.kind = kind
        rng = np.random.Generator(np.random.PCG64(seed))
        lo, hi = (0.02, 0.06) if kind == pkv.KV_E4M3 else (0.04, 0.08)      # INT8: N(0,1) / scale inside +-127
        self.ks = (rng.uniform(lo, hi, size=Hkv) if scales else np.ones(Hkv)).astype(np.float32)
        self.vs = (rng.uniform(lo, hi, size=Hkv) if scales else np.ones(Hkv)).astype(np.float32)
        self.k8, self.v8 = quantize(p.k_cache, self.ks, kind), quantize(p.v_cache, self.vs, kind)
        self.q, self.k, self.v = to_dev(p.q), to_dev(self.k8), to_dev(self.v8)
        self.bt, self.sl = to_dev(p.block_table), to_dev(p.seq_lens)
        self.dks, self.dvs = (to_dev(self.ks), to_dev(self.vs)) if scales else (None, None)
        self.shape = pkv.Shape(B=p.B, Hq=p.Hq, Hkv=Hkv, page_size=page_size, max_pages=p.block_table.shape[1],
                               num_pages=p.k_cache.shape[0], kv_dtype=kind, k_scale=self.dks, v_scale=self.dvs)
        self.out = torch.full((p.B, p.Hq, p.d), float("nan"), dtype=torch.float16, device="cuda")
        self.lse = torch.full((p.B, p.Hq), float("nan"), dtype=torch.float32, device="cuda")

    def oracle(self):
        p = self.p
        return pkv_oracle.attention_fp8(p.q, self.k8, self.v8, self.ks, self.vs, p.block_table, p.seq_lens, Hkv=p.Hkv,
                                        page_size=p.page_size, scale=p.scale, kv_kind=2 if self.kind == pkv.KV_INT8 else 1)

    def decode(self, pol):
        ws = pkv.alloc_workspace(self.shape, pol)
        self.out.fill_(float("nan"))
        self.lse.fill_(float("nan"))
        pkv.pkv_decode(self.shape, pol, self.q, self.k, self.v, self.bt, self.sl, self.out, self.lse, scale=self.p.scale,
                       workspace=ws)
        torch.cuda.synchronize()
        return self.out.cpu().numpy().astype(np.float64), self.lse.cpu().numpy().astype(np.float64), ws


def _check(fp, pol, ref, what):
    out, lse, ws = fp.decode(pol)
    assert not np.isnan(out).any(), what
    assert_within_tolerance(out, ref[0], what)
    fin = np.isfinite(ref[1])
    assert np.array_equal(np.isneginf(lse), np.isneginf(ref[1])), what
    assert np.abs(lse[fin] - ref[1][fin]).max(initial=0.0) <= 2e-3, what
    return ws


@pytest.mark.parametrize("kind", [pkv.KV_E4M3, pkv.KV_INT8])
@pytest.mark.parametrize("Hkv", [8, 4])
@pytest.mark.parametrize("P", [16, 32])
def test_fp8_ragged_sweep(Hkv, P, kind):
    fp = Fp8Problem(RAGGED, seed=1000 + Hkv + P, Hkv=Hkv, page_size=P, kind=kind)
    ref = fp.oracle()
    for hg in (0, 1, 2, 4, 8):
        if hg > Hkv:
            continue
        for pol in (pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=5, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=3, heads_per_cta=hg, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT),
                    pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, heads_per_cta=hg)):
            ws = _check(fp, pol, ref, "fp8 Hkv%d P%d hg%d %s" % (Hkv, P, hg, pol))
    tasks, offs = pkv.pkv_read_workqueue(fp.shape, pol, ws)
    want = wq.build_workqueue(RAGGED, Hkv, oracle_policy(pol))
    assert tasks.tolist() == [list(t) for t in want.tasks]


def test_fp8_unit_scales_dominant_key_and_token_counts():
    """NULL scale pointers mean 1.0; a dominant key at block / tile / split boundaries returns that
    token's (dequantised) V; with K = 0 bytes every output is the mean of V over exactly N tokens."""
    fp = Fp8Problem([1000, 33, 4097], seed=1100, scales=False)
    _check(fp, pkv.Policy(tile_tokens=32, num_splits=4), fp.oracle(), "unit scales")
    S, N = 4, 1000
    c = -(-(-(-N // 32)) // S) * 32
    dec = np.vectorize(pkv_oracle.e4m3_to_double)
    for j in (0, 15, 16, 17, 31, 32, c - 1, c, c + 1, N - 1):
        fj = Fp8Problem([N], seed=1101)
        page, r = int(fj.p.block_table[0, j // 16]), j % 16
        for g in range(8):
            big = np.clip(3.0 * fj.p.q[0, g * 4].astype(np.float32) / fj.ks[g], -448.0, 448.0)
            fj.k8[page, r, g] = torch.from_numpy(big).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
        fj.k = to_dev(fj.k8)
        out, _, _ = fj.decode(pkv.Policy(tile_tokens=32, num_splits=S))
        for g in range(8):
            want = dec(fj.v8[page, r, g]) * fj.vs[g]
            assert np.abs(out[0, g * 4] - want).max() <= 2e-3, (j, g)
    fz = Fp8Problem([4097, 33, 1, 1000], seed=1102)
    fz.k8[...] = 0
    fz.k = to_dev(fz.k8)
    out, lse, _ = fz.decode(pkv.Policy(tile_tokens=32, num_splits=7))
    assert_within_tolerance(out, fz.oracle()[0])
    assert np.allclose(lse, np.log(np.array([4097, 33, 1, 1000], dtype=np.float64))[:, None], atol=1e-5)


@pytest.mark.parametrize("kind", [pkv.KV_E4M3, pkv.KV_INT8])
@pytest.mark.parametrize("Hq,Hkv", [(32, 32), (32, 16), (64, 4), (32, 2)])
def test_fp8_other_group_sizes(Hq, Hkv, kind):
    """One-byte caches with G = 1, 2 and 16 (the paper's GQA sweep, on the caches of
    PAPER.md:271): every heads-per-CTA variant, both routes, separate and fused merge."""
    G = Hq // Hkv
    fp = Fp8Problem(RAGGED, seed=1300 + Hq + Hkv, Hkv=Hkv, Hq=Hq, kind=kind)
    ref = fp.oracle()
    for hg in (0, 1, 2, 4, 8):
        if hg > Hkv or (G == 16 and hg == 8):
            continue
        for pol in (pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=5, heads_per_cta=hg),
                    pkv.Policy(tile_tokens=32, num_splits=3, heads_per_cta=hg, merge_mode=pkv.MERGE_FUSED, route=pkv.ROUTE_RECT),
                    pkv.Policy(tile_tokens=32, split_mode=pkv.SPLIT_BALANCED, num_splits=0, num_sms=24, heads_per_cta=hg)):
            ws = _check(fp, pol, ref, "one-byte G%d Hkv%d hg%d %s" % (G, Hkv, hg, pol))
    tasks, offs = pkv.pkv_read_workqueue(fp.shape, pol, ws)
    want = wq.build_workqueue(RAGGED, Hkv, oracle_policy(pol))
    assert tasks.tolist() == [list(t) for t in want.tasks]


def test_fp8_unsupported_combinations_are_refused():
    fp = Fp8Problem([100], seed=1200)
    with pytest.raises(pkv.PkvError):
        fp.decode(pkv.Policy(tile_tokens=32, num_splits=2, kernel=pkv.KERNEL_SIMT))
    with pytest.raises(pkv.PkvError) as ei:              # one-byte caches: d = 128 only
        pkv.pkv_workspace_partials(pkv.Shape(B=1, Hq=32, Hkv=8, d=64, page_size=16, max_pages=8, num_pages=8, kv_dtype=pkv.KV_E4M3),
                                   pkv.Policy(tile_tokens=32, num_splits=2), torch.zeros(1 << 20, dtype=torch.uint8, device="cuda"))
    assert ei.value.status == pkv.PKV_ERR_UNSUPPORTED


def test_int8_all_byte_values_and_token_counts():
    """INT8 caches: every byte value -128 .. 127 appears in K and V (the in-register int8 -> FP16
    conversion is exact for all of them, so the result matches the oracle as closely as FP16 caches
    do), unit scales through NULL pointers, and the K = 0 counting pin."""
    fp = Fp8Problem([600, 33, 4097], seed=1500, scales=False, kind=pkv.KV_INT8)
    rng = np.random.Generator(np.random.PCG64(4))
    fp.k8 = (rng.integers(-3, 4, size=fp.k8.shape)).astype(np.int8).view(np.uint8)      # small keys: soft attention
    fp.v8 = rng.integers(-128, 128, size=fp.v8.shape).astype(np.int8).view(np.uint8)     # every byte value
    assert len(np.unique(fp.v8)) == 256
    fp.k, fp.v = to_dev(fp.k8), to_dev(fp.v8)
    ref = fp.oracle()
    for pol in (pkv.Policy(tile_tokens=32, num_splits=4), pkv.Policy(tile_tokens=32, num_splits=1, heads_per_cta=2)):
        out, lse, _ = fp.decode(pol)
        assert np.abs(out - ref[0]).max() <= 0.05 and np.abs(out - ref[0]).max() / np.abs(ref[0]).max() <= 2e-3
        assert np.abs(lse - ref[1]).max() <= 2e-3
    fp.k8[...] = 0
    fp.k = to_dev(fp.k8)
    out, lse, _ = fp.decode(pkv.Policy(tile_tokens=32, num_splits=7))
    assert np.allclose(lse, np.log(np.array([600, 33, 4097], dtype=np.float64))[:, None], atol=1e-5)
