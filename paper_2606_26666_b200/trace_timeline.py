"""Timeline of back-to-back decode steps from the library's debug trace hook.

    python -m paper_2606_26666_b200.trace_timeline [--workload config2] [--split-mode 0 --splits 16 --tile-tokens 32]

`pkv_debug_set_trace` makes every decode CTA (and merge CTA) stamp %globaltimer at fixed points of
the kernel.  This captures three steps {decode, merge} in one CUDA graph, as bench.py replays
them, and prints when each phase happens relative to the first decode CTA's start (min / median
/ max over CTAs, microseconds; the timer ticks in 256 ns steps here).  It is how DESIGN.md's
per-step timeline was measured; it is not a benchmark.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DECODE_STAMPS = ["CTA start", "passed griddepcontrol.wait", "first unit known", "first TMA issued", "first K page landed",
                 "first unit: page loop done", "first unit: state stored", "producer done", "plan done"]
MERGE_STAMPS = ["CTA start", "passed griddepcontrol.wait", "states loaded", "output stored"]
MAX_SMS, MERGE_CTAS = 148, 4096


def main():
    import torch

    import paper_2606_26666_b200 as pkv
    import pkv_inputs

    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="config2", choices=["config2", "config3", "config4", "config4_b4"])
    ap.add_argument("--split-mode", type=int, default=pkv.SPLIT_BALANCED)
    ap.add_argument("--splits", type=int, default=0)
    ap.add_argument("--tile-tokens", type=int, default=16)
    ap.add_argument("--seed", type=int, default=pkv_inputs.REPORT_SEEDS[0])
    a = ap.parse_args()
    w = getattr(pkv_inputs, a.workload)(a.seed)
    dev = torch.device("cuda", 0)
    shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, max_pages=w.max_pages, num_pages=w.num_pages)
    pol = pkv.Policy(tile_tokens=a.tile_tokens, split_mode=a.split_mode, num_splits=a.splits)
    R = 3   # one KV pool per step: no step finds its K/V in L2
    qs = [pkv_inputs.fill_pool_torch((w.B, w.Hq, w.d), 1 + r, dev) for r in range(R)]
    ks = [pkv_inputs.fill_pool_torch(w.pool_shape(), 10 + r, dev) for r in range(R)]
    vs = [pkv_inputs.fill_pool_torch(w.pool_shape(), 20 + r, dev) for r in range(R)]
    bt = torch.from_numpy(w.block_table).to(dev)
    sl = torch.from_numpy(w.seq_lens.astype(np.int32)).to(dev)
    out = torch.zeros((w.B, w.Hq, w.d), dtype=torch.float16, device=dev)
    ws = pkv.alloc_workspace(shape, pol)
    traces = [torch.zeros((MAX_SMS * 16 + MERGE_CTAS * 4,), dtype=torch.int64, device=dev) for _ in range(R)]
    st = torch.cuda.Stream()

    def step(r, traced):
        pkv.pkv_debug_set_trace(traces[r].data_ptr() if traced else 0)
        pkv.pkv_decode_stages(shape, pol, qs[r], ks[r], vs[r], bt, sl, out, None, scale=0.0, stages=pkv.STAGE_ALL,
                              workspace=ws, stream=st)

    try:
        with torch.cuda.stream(st):
            for i in range(6):
                step(i % R, False)
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(st):
            with torch.cuda.graph(g, stream=st):
                for r in range(R):
                    step(r, True)
    finally:
        pkv.pkv_debug_set_trace(0)
    for _ in range(3):
        for t in traces:
            t.zero_()
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            g.replay()
        st.synchronize()
    T = [t.cpu().numpy().astype(np.float64) for t in traces]
    d0 = T[0][:MAX_SMS * 16].reshape(MAX_SMS, 16)[:, 0]
    t0 = d0[d0 > 0].min()

    def stat(v):
        v = v[v > 0]
        if not len(v):
            return "-"
        return "min %7.2f  med %7.2f  max %7.2f  (%d CTAs)" % ((v.min() - t0) / 1e3, (np.median(v) - t0) / 1e3,
                                                                (v.max() - t0) / 1e3, len(v))

    c = pkv.pkv_get_counters(shape, pol, ws, stream=st)
    print("workload %s  policy %s  tasks %d  max splits per row %d  chunk_tiles %d" % (
        w.name, pol, c["tasks"], c["max_row_splits"], c["chunk_tiles"]))
    for r in range(R):
        d = T[r][:MAX_SMS * 16].reshape(MAX_SMS, 16)
        m = T[r][MAX_SMS * 16:].reshape(MERGE_CTAS, 4)
        for i, name in enumerate(DECODE_STAMPS):
            print("step %d  decode  %-28s %s" % (r, name, stat(d[:, i])))
        for i, name in enumerate(MERGE_STAMPS):
            print("step %d  merge   %-28s %s" % (r, name, stat(m[:, i])))


if __name__ == "__main__":
    main()
