#!/usr/bin/env python
"""bench.py -- decode tokens/s and achieved HBM GB/s of the PersistentKV hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config2|...]

One "step" is one pass of the whole hot path over one decode batch:
device workqueue builder -> paged GQA decode kernel -> segmented merge, through the C ABI of
include/pkv.h (`pkv_decode`), captured in CUDA graphs.  The headline workload at
N = 1 is BASELINE.json configs[1] (B=1, N=32768, 2048 pages permuted in a 4096-page pool, split
sweep {1,4,16,64} + the auto rule).  DESIGN.md "Measurement" states every definition used here.

What is printed (ONE JSON line, rank 0):
  value      decode tokens/s = (rows decoded by all ranks in K steps) / (max over ranks of the
             CUDA-event time of those K steps), inputs resident in HBM
  e2e        the same through pkv_decode_host with HOST buffers for q / block_table / seq_lens
             / out (host planning + one H2D image + launches + D2H + sync per step), wall clock
  roofline   the decode kernel alone (PKV_STAGE_BUILD|PKV_STAGE_DECODE launches -- one kernel,
             the queue is derived inside it -- back to back between two CUDA events): algorithmic bytes / average launch time / measured HBM peak
  cpu_baseline  oracle/ (FP64, test infrastructure) timed on this box's host cores, rank 0, N = 1
L2: step t uses KV pool t % R of R rotating pools (R * KV bytes per step >> 126 MB L2), so no
step finds its K/V in L2 ("inputs larger than L2").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import pkv_inputs  # noqa: E402  (seeded input generators; no attention arithmetic)

L2_BYTES = 126 * 1000 * 1000
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2",
                    choices=["config1", "config2", "config3", "config4", "config4_b4", "config5", "config5_hkv4"])
    ap.add_argument("--seed", type=int, default=pkv_inputs.REPORT_SEEDS[0])
    ap.add_argument("--hkv", type=int, default=0, help="config3 only: KV heads (GQA sweep, G = 32 / hkv in {1, 2, 4, 8})")
    ap.add_argument("--rotate", type=int, default=0, help="rotating KV pools (0 = enough to exceed L2 4x)")
    ap.add_argument("--tile-tokens", type=int, default=0)
    ap.add_argument("--split-mode", type=int, default=-1)
    ap.add_argument("--splits", type=int, default=-1)
    ap.add_argument("--chunk-tiles", type=int, default=-1)
    ap.add_argument("--route", type=int, default=-1)
    ap.add_argument("--merge", type=int, default=-1)
    ap.add_argument("--kernel", type=int, default=-1)
    ap.add_argument("--hg", type=int, default=0, help="force KV heads per CTA (test hook)")
    ap.add_argument("--graph-steps", type=int, default=100, help="decode steps per CUDA graph (configs[1]: 100)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the split-count sweep / extra workloads")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


# ------------------------------------------------------------------ workload

def make_workload(name: str, seed: int, hkv: int = 0):
    if name == "config1":
        return pkv_inputs.config1(seed)
    if name == "config2":
        return pkv_inputs.config2(seed)
    if name == "config3":
        return pkv_inputs.config3(seed, Hkv=hkv) if hkv else pkv_inputs.config3(seed)
    if name == "config4":
        return pkv_inputs.config4(seed)
    if name == "config4_b4":
        return pkv_inputs.config4_b4(seed)
    if name == "config5":
        return pkv_inputs.config5(seed)
    if name == "config5_hkv4":
        return pkv_inputs.config5(seed, Hkv=4)
    raise ValueError(name)


def algorithmic_bytes(w, lens) -> int:
    """K+V resident for the active rows + q in + out + block-table entries used
    + seq_lens.  Partials, task list and merge traffic are overhead, not roofline bytes."""
    lens = np.asarray(lens, dtype=np.int64)
    kv = int(lens.sum()) * w.kv_bytes_per_token()
    qo = 2 * w.B * w.Hq * w.d * 2
    bt = int(((lens + w.page_size - 1) // w.page_size).sum()) * 4 + w.B * 4
    return kv + qo + bt


def default_policy(pkv, name: str, args):
    """Per-workload default split policy (tuned on seed 20260622)."""
    if name in ("config1",):
        pol = pkv.Policy(tile_tokens=32, num_splits=1, route=pkv.ROUTE_RECT)
    else:
        # BALANCED (A21): chunk from the batch's true lengths, page-granular tiles
        pol = pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, route=pkv.ROUTE_WORKQUEUE)
    if args.tile_tokens > 0:
        pol.tile_tokens = args.tile_tokens
    if args.split_mode >= 0:
        pol.split_mode = args.split_mode
    if args.splits >= 0:
        pol.num_splits = args.splits
    if args.chunk_tiles >= 0:
        pol.chunk_tiles = args.chunk_tiles
    if args.route >= 0:
        pol.route = args.route
    if args.merge >= 0:
        pol.merge_mode = args.merge
    if args.kernel >= 0:
        pol.kernel = args.kernel
    return pol


# ------------------------------------------------------------------ device state and graphs

class Runner:
    """Device-resident state of one workload: R rotating (q, K pool, V pool, block_table) sets, a
    [steps+1, B] table of per-step lengths (N_i += 1 per step, BASELINE.json configs[2..4]), one
    workspace, one output.  PyTorch owns memory, streams and graphs; every step of the path runs
    in libpkv.so."""

    def __init__(self, pkv, torch, w, pol, R, seed, device):
        self.pkv, self.torch, self.w, self.pol, self.R = pkv, torch, w, pol, R
        self.device = device
        self.scale = float(np.float32(1.0 / math.sqrt(w.d)))
        self.shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, d=w.d, page_size=w.page_size,
                               max_pages=w.max_pages, num_pages=w.num_pages)
        self.q, self.k, self.v, self.bt = [], [], [], []
        for r in range(R):
            self.q.append(pkv_inputs.fill_pool_torch((w.B, w.Hq, w.d), seed * 100 + 3 * r + 1, device))
            self.k.append(pkv_inputs.fill_pool_torch(w.pool_shape(), seed * 100 + 3 * r + 2, device))
            self.v.append(pkv_inputs.fill_pool_torch(w.pool_shape(), seed * 100 + 3 * r + 3, device))
            self.bt.append(torch.from_numpy(w.block_table).to(device))
        self.nlens = w.steps + 1
        lens_all = np.stack([w.seq_lens_at(t) for t in range(self.nlens)]).astype(np.int32)
        self.lens_all_host = lens_all
        self.lens_all = torch.from_numpy(lens_all).to(device)
        self.sl = torch.from_numpy(lens_all[0].copy()).to(device)
        self.out = torch.zeros((w.B, w.Hq, w.d), dtype=torch.float16, device=device)
        self.stream = torch.cuda.Stream(device=device)
        self.set_policy(pol)

    def set_policy(self, pol):
        """Switches the split policy: new workspace, captured graphs dropped (pools are kept)."""
        self.pol = pol
        self.graphs = {}
        self.ws = self.pkv.alloc_workspace(self.shape, pol, device=self.device)

    def lens_at(self, t):
        return self.lens_all_host[t % self.nlens]

    def launch_step(self, t, stages, stream):
        """Step t: the chosen stages on pool t % R with the lengths of trace step t % (steps+1)
        (row t of the device-resident [steps+1, B] length table: N_i += 1 per step)."""
        r = t % self.R
        sl = self.lens_all[t % self.nlens] if (stages & self.pkv.STAGE_BUILD) else self.lens_all[0]
        self.pkv.pkv_decode_stages(self.shape, self.pol, self.q[r], self.k[r], self.v[r], self.bt[r], sl,
                                   self.out, None, scale=self.scale, stages=stages, workspace=self.ws,
                                   stream=stream)

    def graph(self, t0, n, stages):
        """CUDA graph of steps t0 .. t0+n-1 (cached)."""
        key = (t0, n, stages)
        if key not in self.graphs:
            torch = self.torch
            g = torch.cuda.CUDAGraph()
            with torch.cuda.stream(self.stream):
                with torch.cuda.graph(g, stream=self.stream):
                    for t in range(t0, t0 + n):
                        self.launch_step(t, stages, torch.cuda.current_stream())
            self.graphs[key] = g
        return self.graphs[key]

    def plan(self, K, chunk):
        """Graph replays covering steps 0..K-1 exactly: [(t0, n), ...] with t0 a multiple of chunk
        reduced modulo lcm(R, nlens)-free bookkeeping: chunks start at step 0 of the rotation."""
        out = []
        full, rem = divmod(K, chunk)
        out += [(0, chunk)] * full
        if rem:
            out.append((0, rem))
        return out

    def run(self, K, chunk, stages):
        """Replays graphs for exactly K steps between two CUDA events on self.stream.  Returns ms."""
        torch = self.torch
        plan = self.plan(K, chunk)
        graphs = [self.graph(t0, n, stages) for (t0, n) in plan]     # capture outside the timed region
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(self.stream):
            e0.record(self.stream)
            for g in graphs:
                g.replay()
            e1.record(self.stream)
        e1.synchronize()
        return e0.elapsed_time(e1)

    def eager_step(self, t, stages=None):
        with self.torch.cuda.stream(self.stream):
            self.launch_step(t, self.pkv.STAGE_ALL if stages is None else stages, self.stream)
        self.stream.synchronize()

    def counters(self):
        return self.pkv.pkv_get_counters(self.shape, self.pol, self.ws, stream=self.stream)


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs
    (the recipe's clocks line, /opt/skills/guides/B200_PROFILING.md, at a finer period)."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}

    def __init__(self, index, period_s=0.002):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reason_bits, self.max_mhz = [], 0, None
        self.stop_flag = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        while not self.stop_flag.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                self.reason_bits |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag.set()
        if self.is_alive():
            self.join(timeout=2.0)
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"], "samples": 0}
        reasons = [name for bit, name in self.REASONS.items() if self.reason_bits & bit]
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(self.samples)}


def physical_gpu_index(torch, local_index):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_index])
        except Exception:
            return local_index
    return local_index


# ------------------------------------------------------------------ oracle legs (CPU)

def host_problem(runner, r=0):
    """Host copies (same bits) of rotation slot r, for the oracle."""
    return (runner.q[r].cpu().numpy(), runner.k[r].cpu().numpy(), runner.v[r].cpu().numpy(),
            np.ascontiguousarray(runner.w.block_table))


def oracle_sample(w, lens, q, k, v, bt, scale, target_s, rows=None):
    """Times oracle/ as it stands on a bounded sample of the workload: whole rows of the batch
    (all heads, all tokens), first a probe row to size the sample, then as many rows/steps as fit
    in about target_s.  Returns (tokens_per_s scaled to the whole batch, description, cores, out)."""
    from oracle import pkv_oracle

    cores = pkv_oracle.max_threads()
    lens = np.asarray(lens, dtype=np.int32)
    order = list(range(w.B)) if rows is None else list(rows)

    def run(sel):
        t0 = time.perf_counter()
        out, _ = pkv_oracle.attention(np.ascontiguousarray(q[sel]), k, v, np.ascontiguousarray(bt[sel]),
                                      np.ascontiguousarray(lens[sel]), Hkv=w.Hkv, page_size=w.page_size, scale=scale)
        return time.perf_counter() - t0, out

    # probe: shortest row, to estimate seconds per token
    i0 = min(order, key=lambda i: lens[i])
    t_probe, _ = run([i0])
    per_tok = t_probe / max(int(lens[i0]), 1)
    # sample rows in batch order until the estimated time reaches the target
    sel, est = [], 0.0
    for i in order:
        c = per_tok * int(lens[i])
        if sel and est + c > target_s:
            break
        sel.append(i)
        est += c
    t_s, out = run(sel)
    reps = 1
    while t_s * (reps + 1) / reps <= target_s and len(sel) == len(order) and reps < 50:   # whole batch fits: repeat steps
        t2, out = run(sel)
        t_s += t2
        reps += 1
    tok_sel = int(lens[sel].sum())
    tok_all = int(lens[order].sum())
    # time of a whole step extrapolated by KV tokens (the oracle's work is linear in them)
    t_step = (t_s / reps) * tok_all / max(tok_sel, 1)
    desc = "%d of %d rows (%d of %d KV tokens) x %d step(s), %.2f s CPU wall; extrapolated by KV tokens" % (
        len(sel), len(order), tok_sel, tok_all, reps, t_s)
    return w.B / t_step, desc, cores, sel, out


def run_reference(args):
    """--impl reference: the oracle (FP64, plain C, OpenMP over (row, kv head)) timed on the host
    cores on the same workload / metric / unit.  Each "step" is a bounded sample (see `sample`)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = make_workload(args.workload, args.seed, args.hkv)
    scale = float(np.float32(1.0 / math.sqrt(w.d)))
    lens = w.seq_lens_at(0)
    # budget: the whole run (K + W steps) within about two minutes
    n_steps = max(1, args.steps + args.warmup)
    per_step_budget = min(10.0, 120.0 / n_steps)
    # a sample = the first n tokens of the longest row, one KV head group... keep it simple and
    # linear: restrict every row to its first `cap` tokens so that one step costs ~per_step_budget
    q = pkv_inputs.fill_normal_f16((w.B, w.Hq, w.d), args.seed * 100 + 1)
    pages_needed = int(w.block_table[w.block_table != pkv_inputs.PAD_PAGE].max()) + 1 if w.B else 1
    from oracle import pkv_oracle
    cores = pkv_oracle.max_threads()
    # calibrate on a small pool: 1 row, 2048 tokens
    probe_pages = 256
    kp = pkv_inputs.fill_normal_f16((probe_pages, w.page_size, w.Hkv, w.d), 11)
    vp = pkv_inputs.fill_normal_f16((probe_pages, w.page_size, w.Hkv, w.d), 12)
    btp = np.arange(probe_pages, dtype=np.int32)[None, :].copy()
    ntok = probe_pages * w.page_size
    t0 = time.perf_counter()
    pkv_oracle.attention(np.ascontiguousarray(q[:1]), kp, vp, btp, np.array([ntok], dtype=np.int32), Hkv=w.Hkv,
                         page_size=w.page_size, scale=scale)
    per_tok = (time.perf_counter() - t0) / ntok          # one row uses Hkv of the threads only
    tok_all = int(lens.astype(np.int64).sum())
    cap_tokens = int(max(w.page_size, min(tok_all, per_step_budget / per_tok)))
    # sample rows' prefixes: distribute cap_tokens over rows proportionally
    frac = min(1.0, cap_tokens / max(tok_all, 1))
    s_lens = np.maximum(1, np.floor(lens * frac)).astype(np.int32)
    # compact page pool holding just the sampled prefixes (same values as a random pool: N(0,1) f16)
    table, universe = pkv_inputs.make_page_table(s_lens, w.page_size, 0.5,
                                                 np.random.Generator(np.random.PCG64(args.seed)))
    k = pkv_inputs.fill_normal_f16((universe, w.page_size, w.Hkv, w.d), args.seed * 100 + 2)
    v = pkv_inputs.fill_normal_f16((universe, w.page_size, w.Hkv, w.d), args.seed * 100 + 3)
    tok_s = int(s_lens.astype(np.int64).sum())

    def step():
        pkv_oracle.attention(q, k, v, table, s_lens, Hkv=w.Hkv, page_size=w.page_size, scale=scale)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    t = time.perf_counter() - t0
    t_step_full = (t / max(args.steps, 1)) * tok_all / max(tok_s, 1)
    value = w.B / t_step_full
    sample = "each step = the first %.4g%% of every row's tokens (%d of %d KV tokens), time scaled by KV tokens" % (
        100.0 * tok_s / max(tok_all, 1), tok_s, tok_all)
    line = {"impl": "reference", "metric": "decode tokens/s", "value": value, "unit": "tokens/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_step_full, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, None, None, args, 1),
            "cpu_baseline": {"value": value, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def workload_config(w, pol, R, args, n_gpus):
    c = {"workload": "%s (BASELINE.json configs; B=%d Hq=%d Hkv=%d d=%d page=%d, rho=%.2f, seed %d)" % (
        w.name, w.B, w.Hq, w.Hkv, w.d, w.page_size, w.hole_frac, w.seed),
         "global_batch": w.B * n_gpus, "seq_lens_step0": [int(x) for x in w.seq_lens[:16]],
         "trace_steps": w.steps, "parallelism": "replicas x%d (no collective; DESIGN.md multi-GPU)" % n_gpus}
    if pol is not None:
        c["policy"] = {k: int(v) for k, v in pol.__dict__.items()}
    if R is not None:
        kvb = int(w.seq_lens.astype(np.int64).sum()) * w.kv_bytes_per_token()
        c["l2"] = "inputs larger than L2: %d rotating KV pools, %.1f MB of K+V per step, %.0f MB before reuse" % (
            R, kvb / 1e6, R * kvb / 1e6)
        c["graph"] = "CUDA graphs of %d decode steps {decode (queue built inside the kernel), merge}" % args.graph_steps
        c["arithmetic"] = "f16 q/K/V and HMMA operands, f32 scores, softmax state and accumulators, f16 out"
    return c


# ------------------------------------------------------------------ the GPU arm

def measured_hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def time_workload(pkv, torch, w, pol, args, device, K, W, want_decode_only=True):
    """Builds the device state, warms up, times K whole steps and K decode-only launches."""
    kvb = int(w.seq_lens.astype(np.int64).sum()) * w.kv_bytes_per_token()
    R = args.rotate if args.rotate > 0 else max(1, min(8, int(math.ceil(4.0 * L2_BYTES / max(kvb, 1)))))
    free_b, _ = torch.cuda.mem_get_info(device)
    pool_b = 2 * int(np.prod(w.pool_shape())) * 2
    R = max(1, min(R, int(free_b * 0.8 // max(pool_b, 1))))
    runner = Runner(pkv, torch, w, pol, R, args.seed, device)
    chunk = max(1, min(args.graph_steps, K))
    for t in range(min(3, max(W, 1))):            # eager warm-up (sets kernel attributes outside capture)
        runner.eager_step(t)
    counters = runner.counters()
    w_left = max(W - 3, 0)
    if w_left:
        runner.run(w_left, chunk, pkv.STAGE_ALL)
    runner.run(chunk, chunk, pkv.STAGE_ALL)        # graph warm-up replay
    ms = runner.run(K, chunk, pkv.STAGE_ALL)
    res = {"runner": runner, "R": R, "ms_total": ms, "counters": counters, "chunk": chunk}
    if want_decode_only:
        dec = pkv.STAGE_BUILD | pkv.STAGE_DECODE     # the decode kernel as the step launches it (fused build)
        runner.run(chunk, chunk, dec)
        res["ms_decode_only"] = runner.run(K, chunk, dec)
    return res


def mean_alg_bytes(w, K, nlens):
    tot = 0
    for t in range(min(K, nlens)):
        tot += algorithmic_bytes(w, w.seq_lens_at(t % nlens))
    n = min(K, nlens)
    return tot / max(n, 1)


def run_e2e(pkv, torch, runner, K, W):
    """K steps through pkv_decode_host: host planning + one H2D image + launches + D2H + sync per
    step, wall clock over the K calls.  KV pools stay resident (the model's state)."""
    w, pol = runner.w, runner.pol
    nb = pkv.pkv_host_scratch_bytes(runner.shape, pol)
    staging = torch.empty(nb, dtype=torch.uint8).pin_memory()
    scratch = torch.empty(nb, dtype=torch.uint8, device=runner.device)
    q_host = [runner.q[r].cpu().pin_memory() for r in range(runner.R)]
    bt_host = torch.from_numpy(np.ascontiguousarray(w.block_table)).pin_memory()
    out_host = torch.empty((w.B, w.Hq, w.d), dtype=torch.float16).pin_memory()
    lens_host = [torch.from_numpy(runner.lens_all_host[t].copy()).pin_memory() for t in range(runner.nlens)]
    c = None

    def step(t):
        r = t % runner.R
        return pkv.pkv_decode_host(runner.shape, pol, q_host[r].data_ptr(), runner.k[r], runner.v[r],
                                   bt_host.data_ptr(), lens_host[t % runner.nlens].data_ptr(), out_host.data_ptr(),
                                   runner.scale, staging, scratch, runner.ws, stream=runner.stream)

    for t in range(max(W, 3)):
        c = step(t)
    torch.cuda.synchronize(runner.device)
    t0 = time.perf_counter()
    for t in range(K):
        c = step(t)
    torch.cuda.synchronize(runner.device)
    dt = time.perf_counter() - t0
    return dt, c, out_host


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2606_26666_b200 as pkv   # raises if libpkv.so is missing: there is no fallback
    from paper_2606_26666_b200 import multirank

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    if args.hg:
        pkv.pkv_debug_force_heads_per_cta(args.hg)
    K, W = args.steps, max(args.warmup, 3)

    # every rank is a replica with its own seeded trace (data-parallel by row; DESIGN.md multi-GPU)
    seed = multirank.rank_seed(args.seed, rank)
    w = make_workload(args.workload, seed, args.hkv)
    pol = default_policy(pkv, args.workload, args)
    peak, peak_src = measured_hbm_peak()

    sweep = {}
    if args.workload == "config2" and not args.no_sweep and args.splits < 0:
        # BASELINE.json configs[1]: split counts {1, 4, 16, 64} (FIXED_COUNT, 32-token tiles), the
        # paper's auto rule (A12) and the BALANCED policy (A21); the timed run uses the fastest
        cands = [(str(S), pkv.Policy(tile_tokens=32, num_splits=S, route=pol.route, merge_mode=pol.merge_mode,
                                     kernel=pol.kernel)) for S in (1, 4, 16, 64, 0)] + [("balanced", pol)]
        # FIXED_COUNT with one single-head unit per SM: S = floor(SMs / (B * Hkv))
        s_fit = torch.cuda.get_device_properties(device).multi_processor_count // max(1, w.B * w.Hkv)
        if s_fit > 1 and s_fit not in (4, 16, 64):
            cands.append((str(s_fit), pkv.Policy(tile_tokens=32, num_splits=s_fit, route=pol.route,
                                                 merge_mode=pol.merge_mode, kernel=pol.kernel)))
        # BALANCED aimed at one unit per SM with 4 / 2 KV heads per CTA: U = SMs * HG / Hkv pairs
        sms = torch.cuda.get_device_properties(device).multi_processor_count
        for hg in (4, 2):
            if w.Hkv % hg == 0 and w.Hkv > hg:
                cands.append(("balanced_hg%d" % hg, pkv.Policy(**{**pol.__dict__, "num_sms": sms * hg // w.Hkv})))
        pols = {}
        for key, p2 in cands:
            r = time_workload(pkv, torch, w, p2, args, device, min(K, 4 * args.graph_steps), W, want_decode_only=False)
            us = 1e3 * r["ms_total"] / min(K, 4 * args.graph_steps)
            if key == "0":
                key = "auto(%d)" % r["counters"]["num_splits"]
            sweep[key] = {"us_per_step": round(us, 3), "tasks": r["counters"]["tasks"],
                          "alg_GBps": round(algorithmic_bytes(w, w.seq_lens) / us / 1e3, 1)}
            pols[key] = p2
            del r
            torch.cuda.empty_cache()
        pol = pols[min(sweep, key=lambda k_: sweep[k_]["us_per_step"])]

    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(device)
    sampler = ClockSampler(physical_gpu_index(torch, local))
    # state + warm-up first, sampling only around the timed calls
    kvb = int(w.seq_lens.astype(np.int64).sum()) * w.kv_bytes_per_token()
    res = time_workload(pkv, torch, w, pol, args, device, min(K, args.graph_steps), W, want_decode_only=False)
    runner = res["runner"]
    chunk = res["chunk"]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(device)
    sampler.start()
    ms_total = runner.run(K, chunk, pkv.STAGE_ALL)
    torch.cuda.synchronize(device)
    if world > 1:
        dist.barrier()
    dec = pkv.STAGE_BUILD | pkv.STAGE_DECODE         # the decode kernel as the step launches it (fused build)
    runner.run(chunk, chunk, dec)
    ms_dec = runner.run(K, chunk, dec)
    clocks = sampler.result()
    counters = res["counters"]

    e2e = None
    if not args.no_e2e:
        dt, c_e2e, _ = run_e2e(pkv, torch, runner, K, W)
        e2e = (dt, c_e2e)

    # max over ranks
    ms_total, ms_dec, e2e_s = multirank.max_over_ranks([ms_total, ms_dec, e2e[0] if e2e else 0.0], device)
    rows_all, = multirank.sum_over_ranks([w.B], device)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    alg = mean_alg_bytes(w, K, runner.nlens)
    us_step = 1e3 * ms_total / K
    us_dec = 1e3 * ms_dec / K
    launches_per_step = counters["build_launches"] + counters["decode_launches"] + counters["merge_launches"]
    line = {
        "metric": "decode tokens/s", "value": multirank.whole_job_tokens_per_s(rows_all, K, ms_total), "unit": "tokens/s",
        "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_total / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f16", "data": "synthetic",
        "config": workload_config(w, pol, res["R"], args, world),
        "us_per_step": us_step,
        "hbm_GBps_whole_step": alg / us_step / 1e3,
        "hbm_frac_whole_step": alg / us_step / 1e3 / peak,
        "launches_per_step": {"build": counters["build_launches"], "decode": counters["decode_launches"],
                              "merge": counters["merge_launches"], "tasks": counters["tasks"],
                              "num_splits": counters["num_splits"], "chunk_tiles": counters["chunk_tiles"],
                              "max_row_splits": counters["max_row_splits"]},
        "gpu_launches": int(launches_per_step * K),
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "pkv_decode_tma_kernel" if pol.kernel != pkv.KERNEL_SIMT else "pkv_decode_simt_kernel",
                     "achieved": alg / us_dec / 1e3, "peak": peak, "unit": "GB/s", "frac": alg / us_dec / 1e3 / peak,
                     "peak_source": peak_src, "frac_of_8TBps_nominal": alg / us_dec / 1e3 / 8000.0,
                     "algorithmic_bytes_per_launch": alg, "us_per_launch": us_dec, "traffic": None},
    }
    if sweep:
        line["config"]["split_sweep"] = sweep
    if e2e:
        c = e2e[1]
        line["e2e"] = {"value": rows_all * K / e2e_s, "unit": "tokens/s", "us_per_step": 1e6 * e2e_s / K,
                       "h2d_bytes_per_step": c["h2d_bytes"], "d2h_bytes_per_step": c["d2h_bytes"],
                       "api": "pkv_decode_host (host planning + 1 H2D + launches + result written to pinned host memory + sync per step)"}

    # parity of the timed configuration + the oracle timed beside it (rank 0, N = 1)
    if world == 1 and not args.no_cpu_baseline:
        q, k, v, bt = host_problem(runner, 0)
        lens = runner.lens_at(0)
        tps, desc, cores, sel, ref = oracle_sample(w, lens, q, k, v, bt, runner.scale, args.cpu_seconds)
        runner.eager_step(0)
        got = runner.out.cpu().numpy().astype(np.float64)[sel]
        err = np.abs(got - ref)
        line["cpu_baseline"] = {"value": tps, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": desc}
        line["parity"] = {"rows_checked": len(sel), "max_abs_err": float(err.max()), "mean_abs_err": float(err.mean()),
                          "tolerance_max_abs": 2e-3, "ok": bool(err.max() <= 2e-3)}
    # traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of the decode kernel from the
    # committed `ncu --set full` capture of this workload (profiles/traffic.csv names the capture)
    traffic_path = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(traffic_path):
        try:
            with open(traffic_path) as f:
                for ln in f:
                    cols = [c.strip() for c in ln.split(",")]
                    if len(cols) >= 3 and cols[0] == args.workload:
                        line["roofline"]["traffic"] = float(cols[2])
                        line["roofline"]["traffic_source"] = cols[3] if len(cols) > 3 else "profiles/traffic.csv"
        except Exception:
            pass
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
