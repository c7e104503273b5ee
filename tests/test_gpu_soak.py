"""Soak: include/pkv.h promises results that are "bitwise reproducible from launch to launch for the
same inputs, policy and device".  Here full-size steps are replayed thousands of times from CUDA
graphs with programmatic dependent launch on -- every kernel overlaps the tail of its predecessor, the
speculative plan and the L2 prefetch run against a predecessor that is still writing -- and every
output must equal the first run's bit for bit.  A race in the stage ring, the workqueue hand-out, the
fused merge's arrival counting or the append patch shows up as a mismatch here long before it shows
up as a tolerance failure (the "stage release" hazard of DESIGN.md 6.1 was found this way).
Element-wise parity with the oracle is the business of the other GPU tests."""
import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
import pkv_inputs as pi
from gpu_helpers import sm_count
from helpers import default_scale

pytestmark = pytest.mark.gpu

PER_GRAPH, REPLAYS = 40, 250         # 10 000 steps per case, about two seconds each


def _rope(npos, d):
    inv = 10000.0 ** (-np.arange(0, d // 2, dtype=np.float64) * 2.0 / d)
    ang = np.arange(npos, dtype=np.float64)[:, None] * inv[None, :]
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)


CASES = [("config2", "auto", "f16", False), ("config2", "balanced", "f16", False), ("config2", "fused16", "f16", False),
         ("config3", "auto", "f16", False), ("config3", "fixed20_hg2", "f16", False), ("config3", "fused20", "f16", False),
         ("config2", "auto", "fp8", False), ("config3", "auto", "int8", False),
         ("config2", "auto", "f16", True), ("config3", "auto", "f16", True), ("config2", "auto", "fp8", True)]


@pytest.mark.parametrize("name,policy,cache,append", CASES)
def test_replayed_steps_are_bitwise_reproducible(name, policy, cache, append):
    dev = torch.device("cuda", 0)
    w = {"config2": pi.config2, "config3": pi.config3}[name](pi.REPORT_SEEDS[2])
    kind = {"f16": pkv.KV_F16, "fp8": pkv.KV_E4M3, "int8": pkv.KV_INT8}[cache]

    def pool(seed):
        t = pi.fill_pool_torch(w.pool_shape(), seed, dev)
        if kind == pkv.KV_E4M3:
            return (t.float() * 32.0).to(torch.float8_e4m3fn).view(torch.uint8)
        if kind == pkv.KV_INT8:
            return (t.float() * 32.0).round().clamp(-127, 127).to(torch.int8).view(torch.uint8)
        return t

    k, v = pool(21), pool(22)
    qs = [pi.fill_pool_torch((w.B, w.Hq, w.d), 23 + i, dev) for i in range(2)]
    bt = torch.from_numpy(w.block_table).to(dev)
    # two alternating steps: different lengths (when the trace grows) and different q
    lens = [w.seq_lens_at(0).astype(np.int32), w.seq_lens_at(min(w.steps, 1)).astype(np.int32)]
    sls = [torch.from_numpy(x).to(dev) for x in lens]
    sc = torch.full((w.Hkv,), 1.0 / 32.0, dtype=torch.float32, device=dev) if kind != pkv.KV_F16 else None
    shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, max_pages=w.max_pages, num_pages=w.num_pages, kv_dtype=kind, k_scale=sc, v_scale=sc)
    if policy == "auto":        # what bench.py times: the cost model's choice
        pol, _ = pkv.pkv_choose_policy(shape, lens[0], pkv.pkv_default_cost_model(sm_count()),
                                       pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_AUTO, num_splits=0))
    else:
        pol = {"balanced": pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0),
               "fused16": pkv.Policy(tile_tokens=32, num_splits=16, merge_mode=pkv.MERGE_FUSED),
               "fused20": pkv.Policy(tile_tokens=32, num_splits=20, merge_mode=pkv.MERGE_FUSED),
               "fixed20_hg2": pkv.Policy(tile_tokens=32, num_splits=20, heads_per_cta=2)}[policy]
    ws = pkv.alloc_workspace(shape, pol)
    out = torch.zeros((w.B, w.Hq, w.d), dtype=torch.float16, device=dev)
    scale = default_scale(w.d)
    app = None
    if append:
        cos, sin = _rope(int(max(x.max() for x in lens)) + 1, w.d)
        app = pkv.Append(k_new=pi.fill_pool_torch((w.B, w.Hkv, w.d), 31, dev), v_new=pi.fill_pool_torch((w.B, w.Hkv, w.d), 32, dev),
                         rope_cos=torch.from_numpy(cos).to(dev), rope_sin=torch.from_numpy(sin).to(dev), rope_positions=cos.shape[0])

    def launch(i, stream):
        if app is not None:       # writes the same bytes to the pool every time
            pkv.pkv_decode_append(shape, pol, qs[i], k, v, bt, sls[i], None, app, out, None, scale=scale, workspace=ws, stream=stream)
        else:
            pkv.pkv_decode(shape, pol, qs[i], k, v, bt, sls[i], out, None, scale=scale, workspace=ws, stream=stream)

    stream = torch.cuda.Stream(device=dev)
    refs = []
    with torch.cuda.stream(stream):
        for i in range(2):
            launch(i, stream)
            launch(i, stream)
            stream.synchronize()
            refs.append(out.clone())
    assert not torch.isnan(refs[0].float()).any() and not torch.equal(refs[0], refs[1])
    hist = torch.zeros((PER_GRAPH,) + tuple(out.shape), dtype=out.dtype, device=dev)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(stream):
        with torch.cuda.graph(g, stream=stream):
            for i in range(PER_GRAPH):
                launch(i % 2, torch.cuda.current_stream())
                hist[i].copy_(out)
    want = torch.stack([refs[i % 2] for i in range(PER_GRAPH)]).view(torch.int16)
    for r in range(REPLAYS):
        with torch.cuda.stream(stream):
            g.replay()
        stream.synchronize()
        neq = (hist.view(torch.int16) != want).flatten(1).any(dim=1)
        assert not bool(neq.any()), "replay %d: steps %s differ from the first run" % (r, torch.nonzero(neq).flatten().tolist()[:8])
    assert pkv.pkv_get_counters(shape, pol, ws, stream=stream)["error_word"] == 0
