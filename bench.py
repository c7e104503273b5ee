#!/usr/bin/env python
"""bench.py -- decode tokens/s and achieved HBM GB/s of the PersistentKV hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config2|...]

One "step" is one pass of the whole hot path over one decode batch:
split-bound policy + workqueue -> paged GQA decode kernel -> segmented merge, through the C ABI of
include/pkv.h (`pkv_decode`), captured in CUDA graphs.  The headline workload at
N = 1 is BASELINE.json configs[1] (B=1, N=32768, 2048 pages permuted in a 4096-page pool, split
sweep {1,4,16,64}).  DESIGN.md "Measurement" states every definition used here.

`--gpus N` without a torchrun environment re-executes itself under `python -m
torch.distributed.run --nproc-per-node N` (one rank per GPU, NCCL); every rank is a replica with
its own seeded trace, there is no data-path collective.

What is printed (ONE JSON line, rank 0):
  value      decode tokens/s = rows decoded by all ranks in K steps / (max over ranks of the
             CUDA-event time of those K steps), inputs resident in HBM.  The K-step region is
             repeated until at least 50 ms have been timed (the first between two synchronizes, the
             others back to back between CUDA events: Runner.run_repeated); value is the MEDIAN
             region, the fastest and the first one are reported beside it (`timing`).
  e2e        the same through pkv_decode_host with HOST buffers for q / block_table / seq_lens
             / out (host planning + H2D + launches + D2H + sync per step), wall clock
  roofline   the decode kernel alone (PKV_STAGE_BUILD|PKV_STAGE_DECODE launches -- one kernel,
             the queue is derived inside it -- back to back between two CUDA events):
             algorithmic bytes / average launch time / measured HBM peak;
             the read-only streaming probe of pkv_calibrate is printed beside the copy peak
  cpu_baseline  oracle/ (FP64, test infrastructure) timed on this box's host cores, rank 0, N = 1
  config.other_workloads  configs 3, 4, 4-B4, 5, 5-Hkv4 and config 3 on the rectangular grid,
             each timed the same way in the same run, with parity against the oracle
Policy: chosen on the TUNE seed 20260622 and frozen; timed on the report seed.
L2: step t uses KV pool t % R of R rotating pools (R * KV bytes per step >> 126 MB L2), so no
step finds its K/V in L2 ("inputs larger than L2").
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import math
import os
import re
import subprocess
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
MIN_TIMED_MS = 50.0                # the K-step region is repeated until this much has been timed
WORKLOADS = ["config1", "config2", "config3", "config4", "config4_b4", "config5", "config5_hkv4", "config2_fp8", "config3_fp8",
             "config2_append", "config3_append", "config2_fp8_append"]
FP8_SCALE = 1.0 / 32.0      # per-KV-head scale of the FP8 workloads: N(0,1) / scale stays far inside +-448


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2", choices=WORKLOADS)
    ap.add_argument("--seed", type=int, default=pkv_inputs.REPORT_SEEDS[0])
    ap.add_argument("--hkv", type=int, default=0, help="config3 only: KV heads (GQA sweep, G = 32 / hkv)")
    ap.add_argument("--rotate", type=int, default=0, help="rotating KV pools (0 = enough to exceed L2 4x)")
    ap.add_argument("--tile-tokens", type=int, default=0)
    ap.add_argument("--split-mode", type=int, default=-1)
    ap.add_argument("--splits", type=int, default=-1)
    ap.add_argument("--chunk-tiles", type=int, default=-1)
    ap.add_argument("--route", type=int, default=-1)
    ap.add_argument("--merge", type=int, default=-1)
    ap.add_argument("--kernel", type=int, default=-1)
    ap.add_argument("--hg", type=int, default=0, help="policy.heads_per_cta (0 = automatic)")
    ap.add_argument("--prefetch-kb", type=int, default=0, help="policy.prefetch_kb (0 = library default, < 0 = off)")
    ap.add_argument("--graph-steps", type=int, default=100, help="decode steps per CUDA graph (configs[1]: 100)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the split-count sweep on the tune seed")
    ap.add_argument("--no-others", action="store_true", help="skip config.other_workloads")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-calibrate", action="store_true", help="skip pkv_calibrate (its probe kernels crowd an ncu launch list)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="target CPU time of the oracle sample")
    ap.add_argument("--timeline", default="", help="write a CUPTI kernel timeline of a few replayed steps to this file")
    ap.add_argument("--timeline-e2e", default="", help="write a CUPTI kernel timeline of a few pipelined host-buffer steps to this file")
    ap.add_argument("--launcher-check", action="store_true",
                    help="exercise only the multi-rank launcher and bookkeeping (gloo, no CUDA): CPU test hook")
    return ap.parse_args(argv)


# ------------------------------------------------------------------ workload

def make_workload(name: str, seed: int, hkv: int = 0):
    if name.endswith("_fp8"):           # the same trace on FP8 (E4M3) caches
        w = make_workload(name[:-4], seed, hkv)
        w.name += "_fp8"
        w.extra["kv_elem_bytes"] = 1
        return w
    if name.endswith("_append"):        # the same trace with the fused KV-append + RoPE step
        w = make_workload(name[:-7], seed, hkv)
        w.name += "_append"
        w.extra["append"] = True
        return w
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


def mean_alg_bytes(w, K, nlens):
    n = max(1, min(K, nlens))
    return sum(algorithmic_bytes(w, w.seq_lens_at(t % nlens)) for t in range(n)) / n


def default_policy(pkv, name: str, args, w=None, num_sms=0):
    """The library's own policy for a workload: config 1 is the paper's unsplit rectangular launch
    (BASELINE.json configs[0] "no splitting"); everything else asks the library's cost model
    (pkv_choose_policy with the default B200 constants on the step-0 lengths, which a serving
    harness has on the host: "for each decode step, the harness estimates T_r").
    Command-line overrides on top (any split override turns the cost model off)."""
    if name in ("config1",):
        pol = pkv.Policy(tile_tokens=32, num_splits=1, route=pkv.ROUTE_RECT)
    else:
        pol = pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, route=pkv.ROUTE_WORKQUEUE)
        if w is not None and num_sms > 0 and args.split_mode < 0 and args.splits < 0 and args.tile_tokens <= 0:
            shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, d=w.d, page_size=w.page_size, max_pages=w.max_pages,
                              num_pages=w.num_pages, kv_dtype=pkv.KV_E4M3 if int(w.extra.get("kv_elem_bytes", 2)) == 1 else pkv.KV_F16)
            base = dataclasses.replace(pol, split_mode=pkv.SPLIT_AUTO)
            pol, _ = pkv.pkv_choose_policy(shape, w.seq_lens, pkv.pkv_default_cost_model(num_sms), base)
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
    if args.hg:
        pol.heads_per_cta = args.hg
    if args.prefetch_kb != 0:
        pol.prefetch_kb = args.prefetch_kb
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
        self.fp8 = int(w.extra.get("kv_elem_bytes", 2)) == 1
        self.kv_scale = torch.full((w.Hkv,), FP8_SCALE, dtype=torch.float32, device=device) if self.fp8 else None
        self.shape = pkv.Shape(B=w.B, Hq=w.Hq, Hkv=w.Hkv, d=w.d, page_size=w.page_size,
                               max_pages=w.max_pages, num_pages=w.num_pages, kv_dtype=pkv.KV_E4M3 if self.fp8 else pkv.KV_F16,
                               k_scale=self.kv_scale, v_scale=self.kv_scale)
        self.q, self.k, self.v, self.bt = [], [], [], []

        def pool(sd):
            t = pkv_inputs.fill_pool_torch(w.pool_shape(), sd, device)
            if not self.fp8:
                return t
            # the same N(0,1) draw, quantised to E4M3 bytes (inputs, not outputs: the oracle gets these bytes)
            return (t.float() / FP8_SCALE).to(torch.float8_e4m3fn).view(torch.uint8)

        for r in range(R):
            self.q.append(pkv_inputs.fill_pool_torch((w.B, w.Hq, w.d), seed * 100 + 3 * r + 1, device))
            self.k.append(pool(seed * 100 + 3 * r + 2))
            self.v.append(pool(seed * 100 + 3 * r + 3))
            self.bt.append(torch.from_numpy(w.block_table).to(device))
        self.nlens = w.steps + 1
        lens_all = np.stack([w.seq_lens_at(t) for t in range(self.nlens)]).astype(np.int32)
        self.lens_all_host = lens_all
        self.lens_all = torch.from_numpy(lens_all).to(device)
        self.out = torch.zeros((w.B, w.Hq, w.d), dtype=torch.float16, device=device)
        self.stream = torch.cuda.Stream(device=device)
        self.buckets = None
        self.append = None
        if w.extra.get("append"):
            # the new token of every row (the same draw every step) and the RoPE tables of a serving engine
            npos = int(lens_all.max()) + 1
            inv = 10000.0 ** (-np.arange(0, w.d // 2, dtype=np.float64) * 2.0 / w.d)
            ang = np.arange(npos, dtype=np.float64)[:, None] * inv[None, :]
            self.rope_host = (np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32))
            self.knew = pkv_inputs.fill_pool_torch((w.B, w.Hkv, w.d), seed * 100 + 91, device)
            self.vnew = pkv_inputs.fill_pool_torch((w.B, w.Hkv, w.d), seed * 100 + 92, device)
            self.append = pkv.Append(k_new=self.knew, v_new=self.vnew, rope_cos=torch.from_numpy(self.rope_host[0]).to(device),
                                     rope_sin=torch.from_numpy(self.rope_host[1]).to(device), rope_positions=npos)
        self.set_policy(pol)

    def set_bucket_route(self, gran):
        """Length-bucket route (pkv_decode_buckets): per trace step the host plan of
        pkv_plan_buckets_host (row index on the device, bucket offsets on the host).  None = off."""
        self.graphs = {}
        if gran is None:
            self.buckets = None
            return
        plans = [self.pkv.pkv_plan_buckets_host(self.lens_all_host[t], gran) for t in range(self.nlens)]
        self.buckets = [(self.torch.from_numpy(ix.copy()).to(self.device), offs.copy()) for ix, offs, _ in plans]
        self.bucket_gran = gran

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
        if self.buckets is not None:
            ix, offs = self.buckets[t % self.nlens]
            self.pkv.pkv_decode_buckets(self.shape, self.pol, self.q[r], self.k[r], self.v[r], self.bt[r],
                                        self.lens_all[t % self.nlens], ix, offs, self.out, None, scale=self.scale,
                                        workspace=self.ws, stream=stream)
            return
        if self.append is not None:
            self.pkv.pkv_decode_append(self.shape, self.pol, self.q[r], self.k[r], self.v[r], self.bt[r],
                                       self.lens_all[t % self.nlens], None, self.append, self.out, None, scale=self.scale,
                                       workspace=self.ws, stream=stream)
            return
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

    def run(self, K, chunk, stages):
        """Replays graphs for EXACTLY K steps between two CUDA events on self.stream.  Returns ms."""
        torch = self.torch
        full, rem = divmod(K, chunk)
        plan = [(0, chunk)] * full + ([(0, rem)] if rem else [])
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

    def run_repeated(self, K, chunk, stages, min_ms=MIN_TIMED_MS, max_regions=400):
        """The exactly-K-step region again and again until min_ms have been timed.  The first region
        is bracketed by a synchronize on both sides (self.run); the others are enqueued back to back,
        each between two CUDA events recorded on the launching stream, with one synchronize after
        the last -- a decode loop in steady state, without a pipeline drain and a graph-launch
        latency inside every K-step region.  Returns the list of region times (ms), first one first."""
        torch = self.torch
        first = self.run(K, chunk, stages)
        n = int(min(max_regions - 1, max(0, math.ceil((min_ms - first) / max(first, 1e-6)))))
        if n == 0:
            return [first]
        full, rem = divmod(K, chunk)
        graphs = [self.graph(t0, m, stages) for (t0, m) in [(0, chunk)] * full + ([(0, rem)] if rem else [])]
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        with torch.cuda.stream(self.stream):
            ev[0].record(self.stream)
            for i in range(n):
                for g in graphs:
                    g.replay()
                ev[i + 1].record(self.stream)
        ev[n].synchronize()
        return [first] + [ev[i].elapsed_time(ev[i + 1]) for i in range(n)]

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

    def __init__(self, index, period_s=0.001):
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


def physical_gpu_index(local_index):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_index])
        except Exception:
            return local_index
    return local_index


def measured_hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def rotation(torch, w, args, device):
    """Rotating KV pools: enough that R * (K+V bytes of a step) exceeds L2 four times over."""
    kvb = int(w.seq_lens.astype(np.int64).sum()) * w.kv_bytes_per_token()
    R = args.rotate if args.rotate > 0 else max(1, min(8, int(math.ceil(4.0 * L2_BYTES / max(kvb, 1)))))
    free_b, _ = torch.cuda.mem_get_info(device)
    pool_b = 2 * int(np.prod(w.pool_shape())) * 2
    return max(1, min(R, int(free_b * 0.8 // max(pool_b, 1))))


def warm(pkv, runner, chunk, W):
    """W warm-up steps: three eager ones (kernel attributes are set outside capture), the rest and
    one more whole graph as replays."""
    for t in range(min(3, max(W, 1))):
        runner.eager_step(t)
    counters = runner.counters()
    if W > 3:
        runner.run(W - 3, chunk, pkv.STAGE_ALL)
    runner.run(chunk, chunk, pkv.STAGE_ALL)
    return counters


def time_policy(pkv, runner, pol, K, chunk, W, decode_only=True):
    """Times one policy on an existing runner: K-step regions (repeated to >= 50 ms) of whole
    steps and of the decode kernel alone.  Returns a dict of region-time lists and counters."""
    runner.set_policy(pol)
    counters = warm(pkv, runner, chunk, W)
    res = {"step_ms": runner.run_repeated(K, chunk, pkv.STAGE_ALL), "counters": counters}
    if decode_only:
        dec = pkv.STAGE_BUILD | pkv.STAGE_DECODE     # the decode kernel as the step launches it (fused build)
        runner.run(chunk, chunk, dec)
        res["decode_ms"] = runner.run_repeated(K, chunk, dec)
    return res


# ------------------------------------------------------------------ oracle legs (CPU; bench.py may execute oracle/ here only)

def host_threads():
    """Threads the oracle is given: the cores this process may run on (torchrun exports
    OMP_NUM_THREADS=1 to its ranks, which would otherwise pin the oracle to one core)."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except Exception:
        return max(1, os.cpu_count() or 1)


def compact_rows(torch, w, k_dev, v_dev, rows, lens):
    """Host copy (same bits) of the pages of `rows` only: compact pools + identity block tables."""
    P = w.page_size
    tables, ks, vs, base = [], [], [], 0
    width = max(1, max(-(-int(lens[i]) // P) for i in rows))
    for i in rows:
        npg = -(-int(lens[i]) // P)
        pages = torch.from_numpy(w.block_table[i, :npg].astype(np.int64)).to(k_dev.device)
        ks.append(k_dev[pages].cpu().numpy())
        vs.append(v_dev[pages].cpu().numpy())
        t = np.full(width, pkv_inputs.PAD_PAGE, dtype=np.int32)
        t[:npg] = np.arange(base, base + npg, dtype=np.int32)
        tables.append(t)
        base += npg
    return np.concatenate(ks), np.concatenate(vs), np.stack(tables)


def oracle_rows(torch, runner, rows, lens, r=0):
    """oracle/ on whole rows of rotation slot r.  Returns (out f64 [len(rows), Hq, d], seconds)."""
    from oracle import pkv_oracle
    w = runner.w
    kc, vc, tc = compact_rows(torch, w, runner.k[r], runner.v[r], rows, lens)
    q = np.ascontiguousarray(runner.q[r].cpu().numpy()[rows])
    sl = np.ascontiguousarray(np.asarray(lens, dtype=np.int32)[rows])
    t0 = time.perf_counter()
    if runner.append is not None:
        from oracle import append_oracle
        kn = np.ascontiguousarray(runner.knew.cpu().numpy()[rows])
        vn = np.ascontiguousarray(runner.vnew.cpu().numpy()[rows])
        if runner.fp8:      # the new token is quantised inside the step (reading A30)
            sc = np.full(w.Hkv, FP8_SCALE, dtype=np.float32)
            out, _, _, _ = append_oracle.append_and_attend_q8(q, kc, vc, sc, sc, kn, vn, tc, sl, runner.rope_host[0], runner.rope_host[1],
                                                               Hkv=w.Hkv, page_size=w.page_size, scale=runner.scale, kv_kind=1)
        else:
            out, _, _, _ = append_oracle.append_and_attend(q, kc, vc, kn, vn, tc, sl, runner.rope_host[0], runner.rope_host[1],
                                                            Hkv=w.Hkv, page_size=w.page_size, scale=runner.scale)
    elif runner.fp8:
        sc = np.full(w.Hkv, FP8_SCALE, dtype=np.float64)
        out, _ = pkv_oracle.attention_fp8(q, kc, vc, sc, sc, tc, sl, Hkv=w.Hkv, page_size=w.page_size, scale=runner.scale,
                                          num_threads=host_threads())
    else:
        out, _ = pkv_oracle.attention(q, kc, vc, tc, sl, Hkv=w.Hkv, page_size=w.page_size, scale=runner.scale,
                                      num_threads=host_threads())
    return out, time.perf_counter() - t0


def pick_rows(lens, budget_tokens, seed):
    """Rows for a bounded oracle check: the shortest and the longest, then seeded random rows while
    the KV-token budget lasts (all rows when they fit)."""
    lens = np.asarray(lens, dtype=np.int64)
    B = len(lens)
    order = [int(np.argmin(lens)), int(np.argmax(lens))]
    rng = np.random.Generator(np.random.PCG64(seed))
    order += [int(i) for i in rng.permutation(B)]
    sel, tok = [], 0
    for i in order:
        if i in sel or lens[i] <= 0:
            continue
        if sel and tok + lens[i] > budget_tokens:
            continue
        sel.append(i)
        tok += int(lens[i])
    return sorted(sel)


def parity_of(torch, runner, rows, t=0):
    """GPU whole step t (eager, the timed policy) against the oracle on `rows`."""
    lens = runner.lens_at(t)
    ref, secs = oracle_rows(torch, runner, rows, lens, r=t % runner.R)
    runner.eager_step(t)
    got = runner.out.cpu().numpy().astype(np.float64)[rows]
    err = np.abs(got - ref)
    tau = np.abs(ref).max(axis=-1, keepdims=True) / 16.0
    rel = err / np.maximum(np.abs(ref), np.maximum(tau, 1e-30))
    ok = bool(err.max() <= 2e-3 and rel.max() <= 1e-2 and not np.isnan(got).any())
    return {"rows_checked": len(rows), "kv_tokens_checked": int(np.asarray(lens)[rows].sum()),
            "max_abs_err": float(err.max()), "mean_abs_err": float(err.mean()), "max_rel_err_floored": float(rel.max()),
            "tolerance": "max abs 2e-3, floored max rel 1e-2 (DESIGN.md A15)", "ok": ok}, secs


def cpu_baseline_of(torch, runner, target_s):
    """oracle/ as it stands, timed on this box's host cores on a bounded sample of the workload:
    whole rows (all heads, all tokens) in seeded order until about target_s of CPU time."""
    from oracle import pkv_oracle
    w = runner.w
    lens = np.asarray(runner.lens_at(0), dtype=np.int64)
    cores = host_threads()
    i0 = int(np.argmin(np.where(lens > 0, lens, lens.max() + 1)))
    _, t_probe = oracle_rows(torch, runner, [i0], lens)
    per_tok = t_probe / max(int(lens[i0]), 1)
    rows = pick_rows(lens, max(int(lens[i0]), int(target_s / max(per_tok, 1e-12))), runner.w.seed)
    reps, t_s = 0, 0.0
    while True:
        _, t1 = oracle_rows(torch, runner, rows, lens)
        t_s += t1
        reps += 1
        if len(rows) < int((lens > 0).sum()) or t_s * (reps + 1) / reps > target_s or reps >= 50:
            break
    tok_sel, tok_all = int(lens[rows].sum()), int(lens.sum())
    t_step = (t_s / reps) * tok_all / max(tok_sel, 1)     # the oracle's work is linear in KV tokens
    desc = "%d of %d rows (%d of %d KV tokens) x %d step(s), %.2f s CPU wall; scaled to a whole step by KV tokens" % (
        len(rows), w.B, tok_sel, tok_all, reps, t_s)
    return {"value": w.B / t_step, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": desc}


def run_reference(args):
    """--impl reference: the oracle (FP64, plain C, OpenMP over (row, kv head)) timed on the host
    cores on the same workload / metric / unit.  Each "step" is a bounded sample (see `sample`).
    Under torchrun rank 0 alone runs it."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import pkv_oracle
    w = make_workload(args.workload, args.seed, args.hkv)
    scale = float(np.float32(1.0 / math.sqrt(w.d)))
    lens = w.seq_lens_at(0)
    n_steps = max(1, args.steps + args.warmup)
    per_step_budget = min(10.0, 120.0 / n_steps)      # the whole run within about two minutes
    q = pkv_inputs.fill_normal_f16((w.B, w.Hq, w.d), args.seed * 100 + 1)
    cores = host_threads()
    probe_pages = 256                                  # calibrate: 1 row, 4096 tokens
    kp = pkv_inputs.fill_normal_f16((probe_pages, w.page_size, w.Hkv, w.d), 11)
    vp = pkv_inputs.fill_normal_f16((probe_pages, w.page_size, w.Hkv, w.d), 12)
    btp = np.arange(probe_pages, dtype=np.int32)[None, :].copy()
    ntok = probe_pages * w.page_size
    t0 = time.perf_counter()
    pkv_oracle.attention(np.ascontiguousarray(q[:1]), kp, vp, btp, np.array([ntok], dtype=np.int32), Hkv=w.Hkv,
                         page_size=w.page_size, scale=scale, num_threads=cores)
    per_tok = (time.perf_counter() - t0) / ntok
    tok_all = int(lens.astype(np.int64).sum())
    cap_tokens = int(max(w.page_size, min(tok_all, per_step_budget / per_tok)))
    frac = min(1.0, cap_tokens / max(tok_all, 1))
    s_lens = np.maximum(1, np.floor(lens * frac)).astype(np.int32)      # every row's first tokens
    table, universe = pkv_inputs.make_page_table(s_lens, w.page_size, 0.5,
                                                 np.random.Generator(np.random.PCG64(args.seed)))
    k = pkv_inputs.fill_normal_f16((universe, w.page_size, w.Hkv, w.d), args.seed * 100 + 2)
    v = pkv_inputs.fill_normal_f16((universe, w.page_size, w.Hkv, w.d), args.seed * 100 + 3)
    tok_s = int(s_lens.astype(np.int64).sum())

    def step():
        pkv_oracle.attention(q, k, v, table, s_lens, Hkv=w.Hkv, page_size=w.page_size, scale=scale, num_threads=cores)

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


# ------------------------------------------------------------------ e2e, timeline, the other workloads

def run_e2e(pkv, torch, runner, K, W, auto=False):
    """K steps through pkv_decode_host: host planning + H2D + launches + D2H + sync per step, wall
    clock over the K calls.  KV pools stay resident (the model's state).  auto: the policy is
    PKV_SPLIT_AUTO, i.e. the cost model runs inside every call on that step's lengths."""
    w = runner.w
    pol = dataclasses.replace(runner.pol, flags=runner.pol.flags | pkv.FLAG_OUT_PINNED)    # out_host below is pinned for good
    ws = runner.ws
    if auto:
        pol = dataclasses.replace(pol, split_mode=pkv.SPLIT_AUTO, num_splits=0)
        ws = pkv.alloc_workspace(runner.shape, pol, device=runner.device)
    nb = pkv.pkv_host_scratch_bytes(runner.shape, pol)
    # one (staging, scratch) pair per rotating KV pool: the pair holds that pool's block table
    staging = [torch.zeros(nb, dtype=torch.uint8).pin_memory() for _ in range(runner.R)]
    scratch = [torch.empty(nb, dtype=torch.uint8, device=runner.device) for _ in range(runner.R)]
    q_host = [runner.q[r].cpu().pin_memory() for r in range(runner.R)]
    bt_host = torch.from_numpy(np.ascontiguousarray(w.block_table)).pin_memory()
    out_host = torch.empty((w.B, w.Hq, w.d), dtype=torch.float16).pin_memory()
    lens_host = [torch.from_numpy(runner.lens_all_host[t].copy()).pin_memory() for t in range(runner.nlens)]
    # the public API a serving loop uses: pkv.HostDecoder (one ctypes call into pkv_decode_host per step)
    dec = [pkv.HostDecoder(runner.shape, pol, runner.k[r], runner.v[r], staging[r], scratch[r], ws, runner.scale,
                           stream=runner.stream) for r in range(runner.R)]
    qp = [q_host[r].data_ptr() for r in range(runner.R)]
    lp = [x.data_ptr() for x in lens_host]
    btp, outp, R, nl = bt_host.data_ptr(), out_host.data_ptr(), runner.R, runner.nlens

    def step(t):
        dec[t % R](qp[t % R], btp, lp[t % nl], outp)

    for t in range(max(W, 3)):
        step(t)
    torch.cuda.synchronize(runner.device)
    t0 = time.perf_counter()
    for t in range(K):
        step(t)
    c = dec[(K - 1) % R].counters
    torch.cuda.synchronize(runner.device)
    return time.perf_counter() - t0, c


def run_e2e_pipelined(pkv, torch, runner, K, W, auto=False):
    """The same K steps through pkv_decode_host_pipelined (pkv.PipelinedHostDecoder): every call is told
    the NEXT step's lengths and block table (a decode loop knows them when it schedules), so the next
    step's launches are enqueued behind a gate while the GPU works on the current one, and a step costs
    a copy of q into pinned memory, a flag store and a spin on the done word.  Same bytes per step over
    the host link, same kernels, bit-identical results (tests/test_gpu_pipelined.py).  One (staging,
    scratch) pair; the rotating KV pools are passed per step.  Returns (seconds, counters, armed fraction)."""
    w = runner.w
    pol = dataclasses.replace(runner.pol, flags=runner.pol.flags | pkv.FLAG_OUT_PINNED)
    ws = runner.ws
    if auto:
        pol = dataclasses.replace(pol, split_mode=pkv.SPLIT_AUTO, num_splits=0)
        ws = pkv.alloc_workspace(runner.shape, pol, device=runner.device)
    nb = pkv.pkv_host_scratch_bytes(runner.shape, pol)
    staging = torch.zeros(nb, dtype=torch.uint8).pin_memory()
    scratch = torch.empty(nb, dtype=torch.uint8, device=runner.device)
    q_host = [runner.q[r].cpu().pin_memory() for r in range(runner.R)]
    bt_host = torch.from_numpy(np.ascontiguousarray(w.block_table)).pin_memory()
    out_host = torch.empty((w.B, w.Hq, w.d), dtype=torch.float16).pin_memory()
    lens_host = [torch.from_numpy(runner.lens_all_host[t].copy()).pin_memory() for t in range(runner.nlens)]
    torch.cuda.synchronize(runner.device)       # nothing may wait for the device once a step is armed
    dec = pkv.PipelinedHostDecoder(runner.shape, pol, runner.k[0], runner.v[0], staging, scratch, ws, runner.scale, stream=runner.stream)
    qp, lp = [x.data_ptr() for x in q_host], [x.data_ptr() for x in lens_host]
    kp, vp = [x.data_ptr() for x in runner.k], [x.data_ptr() for x in runner.v]
    btp, outp, R, nl = bt_host.data_ptr(), out_host.data_ptr(), runner.R, runner.nlens

    # a decode loop passes the same few buffers again and again: marshal each distinct step once
    period = R * nl // math.gcd(R, nl)
    prepared = [dec.prepare(qp[t % R], btp, lp[t % nl], outp, lp[(t + 1) % nl], btp, kp[t % R], vp[t % R], kp[(t + 1) % R], vp[(t + 1) % R])
                for t in range(period)] if period <= 4096 else None
    run = dec.run

    def step(t):
        if prepared is not None:
            run(prepared[t % period])
            return
        r, rn = t % R, (t + 1) % R
        dec(qp[r], btp, lp[t % nl], outp, lp[(t + 1) % nl], btp, kp[r], vp[r], kp[rn], vp[rn])

    try:
        W = max(W, 3)
        for t in range(W):
            step(t)
        t0 = time.perf_counter()
        for t in range(W, W + K):
            step(t)
        dt = time.perf_counter() - t0
        c = dec.counters
        armed, n = 0, min(K, 100)
        for t in range(W + K, W + K + n):       # untimed: how many steps had been enqueued a call early
            step(t)
            armed += int(dec._counters.armed_step)
    finally:
        dec.drain()
    torch.cuda.synchronize(runner.device)
    return dt, c, armed / float(n)


def write_timeline(torch, pkv, runner, path, steps=6):
    """CUPTI (torch.profiler) kernel records of one replay of a `steps`-step graph with programmatic
    dependent launch on: start, duration and the gap to the end of the previous kernel (negative =
    the kernel was resident before its predecessor finished).  Evidence for the CUDA-event numbers
    that ncu cannot give (ncu serialises kernels and removes the overlap)."""
    from torch.profiler import ProfilerActivity, profile
    g = runner.graph(0, steps, pkv.STAGE_ALL)
    with torch.cuda.stream(runner.stream):
        g.replay()
    torch.cuda.synchronize(runner.device)
    with profile(activities=[ProfilerActivity.CUDA]) as prof:
        with torch.cuda.stream(runner.stream):
            g.replay()
            g.replay()
        torch.cuda.synchronize(runner.device)
    evs = [e for e in prof.events() if "pkv_" in e.name]
    evs.sort(key=lambda e: e.time_range.start)
    lines = ["# CUPTI kernel timeline: %s, policy %s" % (runner.w.name, runner.pol),
             "# command: python bench.py --workload %s --timeline <this file> (two replays of a %d-step graph; PDL on)" % (
                 runner.w.name.split("_")[0], steps),
             "# times in microseconds after the first kernel's start; gap = start - end of the previous kernel",
             "%-4s %-34s %10s %10s %10s" % ("#", "kernel", "start", "duration", "gap")]
    if evs:
        t0, prev_end = evs[0].time_range.start, None
        for i, e in enumerate(evs):
            s, d = e.time_range.start - t0, e.time_range.end - e.time_range.start
            gap = "" if prev_end is None else "%10.2f" % (e.time_range.start - prev_end)
            m = re.search(r"pkv_\w+", e.name)
            lines.append("%-4d %-34s %10.2f %10.2f %10s" % (i, m.group(0) if m else e.name[:34], s, d, gap))
            prev_end = e.time_range.end
        n = len(evs) // 2
        span = evs[-1].time_range.end - evs[n].time_range.start
        lines.append("# second replay: %d kernels in %.2f us = %.2f us per step" % (len(evs) - n, span, span / steps))
    with open(path, "w") as f:
        f.write("\n".join(lines) + "\n")


def write_timeline_e2e(torch, pkv, runner, path, steps=8, auto=False):
    """CUPTI (torch.profiler) kernel records of `steps` consecutive steps through pkv.PipelinedHostDecoder, after
    warm-up: per step the gate / stage kernel (its duration includes the time it waits for the host's flag:
    the host's think time plus the flag's way over the host link), decode, merge and the signal kernel.
    Evidence for the e2e wall-clock number; the pipeline is drained before the profiler stops."""
    from torch.profiler import ProfilerActivity, profile
    w = runner.w
    pol = dataclasses.replace(runner.pol, flags=runner.pol.flags | pkv.FLAG_OUT_PINNED)
    ws = runner.ws
    if auto:
        pol = dataclasses.replace(pol, split_mode=pkv.SPLIT_AUTO, num_splits=0)
        ws = pkv.alloc_workspace(runner.shape, pol, device=runner.device)
    nb = pkv.pkv_host_scratch_bytes(runner.shape, pol)
    staging = torch.zeros(nb, dtype=torch.uint8).pin_memory()
    scratch = torch.empty(nb, dtype=torch.uint8, device=runner.device)
    q_host = [runner.q[r].cpu().pin_memory() for r in range(runner.R)]
    bt_host = torch.from_numpy(np.ascontiguousarray(w.block_table)).pin_memory()
    out_host = torch.empty((w.B, w.Hq, w.d), dtype=torch.float16).pin_memory()
    lens_host = [torch.from_numpy(runner.lens_all_host[t].copy()).pin_memory() for t in range(runner.nlens)]
    torch.cuda.synchronize(runner.device)
    dec = pkv.PipelinedHostDecoder(runner.shape, pol, runner.k[0], runner.v[0], staging, scratch, ws, runner.scale, stream=runner.stream)
    R, nl = runner.R, runner.nlens

    def step(t):
        r, rn = t % R, (t + 1) % R
        dec(q_host[r].data_ptr(), bt_host.data_ptr(), lens_host[t % nl].data_ptr(), out_host.data_ptr(), lens_host[(t + 1) % nl].data_ptr(),
            bt_host.data_ptr(), runner.k[r].data_ptr(), runner.v[r].data_ptr(), runner.k[rn].data_ptr(), runner.v[rn].data_ptr())

    walls = []
    try:
        for t in range(20):
            step(t)
        dec.drain()
        with profile(activities=[ProfilerActivity.CUDA]) as prof:
            for t in range(20, 24):          # inside the profiler: first steps re-warm its hooks
                step(t)
            for t in range(24, 24 + steps):
                t0 = time.perf_counter()
                step(t)
                walls.append(1e6 * (time.perf_counter() - t0))
            dec.drain()
            torch.cuda.synchronize(runner.device)
    finally:
        dec.drain()
    evs = [e for e in prof.events() if "pkv_" in e.name]
    evs.sort(key=lambda e: e.time_range.start)
    per_step = 4 if any("pkv_merge" in e.name for e in evs) else 3
    evs = evs[-(steps + 1) * per_step:-per_step]      # the timed steps (the last group is the drained, discarded step)
    lines = ["# CUPTI kernel timeline of %d consecutive pipelined host-buffer steps: %s, policy %s" % (steps, w.name, pol),
             "# command: python bench.py --workload %s --timeline-e2e <this file> (pkv.PipelinedHostDecoder; under the profiler)" % w.name.split("_")[0],
             "# times in microseconds after the first listed kernel's start; gap = start - end of the previous kernel (negative: resident early)",
             "# pkv_stage_kernel is the gate: it starts when the previous step has finished and its duration includes the wait for the host's flag",
             "# wall clock of these calls under the profiler, us: " + " ".join("%.1f" % x for x in walls),
             "%-4s %-34s %10s %10s %10s" % ("#", "kernel", "start", "duration", "gap")]
    if evs:
        t0, prev_end = evs[0].time_range.start, None
        for i, e in enumerate(evs):
            s_, d_ = e.time_range.start - t0, e.time_range.end - e.time_range.start
            gap = "" if prev_end is None else "%10.2f" % (e.time_range.start - prev_end)
            m = re.search(r"pkv_\w+", e.name)
            lines.append("%-4d %-34s %10.2f %10.2f %10s" % (i, m.group(0) if m else e.name[:34], s_, d_, gap))
            prev_end = e.time_range.end
        span = evs[-1].time_range.end - evs[0].time_range.start
        lines.append("# %d kernels in %.2f us = %.2f us per step from gate start to signal end (host think time between steps included)" % (
            len(evs), span, span / steps))
    with open(path, "w") as f:
        f.write("\n".join(lines) + "\n")


def summarize(regions_ms, K):
    us = [1e3 * m / K for m in regions_ms]
    return {"regions": len(us), "us_per_step_median": float(np.median(us)), "us_per_step_min": float(min(us)),
            "us_per_step_max": float(max(us)), "timed_ms_total": float(sum(regions_ms))}


def other_workloads(pkv, torch, args, device, peak, read_peak):
    """configs 3, 4, 4-B4, 5, 5-Hkv4 with the library's own policy, and config 3 on the rectangular
    (B, Hkv, S) grid against the workqueue at the same fixed split count (BASELINE.json configs[2],
    PAPER.md:71, 204-206): us/step (median of >= 50 ms of K-step regions), roofline fraction of the
    decode kernel, launches per step, parity against the oracle on seeded rows."""
    out = {}
    bal = None      # None: the cost model's choice for the workload (default_policy)
    cases = [("config3", "config3", bal),
             ("config3_workqueue_S20", "config3", pkv.Policy(tile_tokens=32, num_splits=20, route=pkv.ROUTE_WORKQUEUE,
                                                             prefetch_kb=args.prefetch_kb)),
             ("config3_rect_S20", "config3", pkv.Policy(tile_tokens=32, num_splits=20, route=pkv.ROUTE_RECT,
                                                        prefetch_kb=args.prefetch_kb)),
             ("config3_buckets_exact_S32", "config3", pkv.Policy(tile_tokens=32, num_splits=32, route=pkv.ROUTE_RECT,
                                                                 prefetch_kb=args.prefetch_kb)),
             ("config4", "config4", bal), ("config4_b4", "config4_b4", bal),
             ("config5", "config5", bal), ("config5_hkv4", "config5_hkv4", bal),
             ("config2_fp8", "config2_fp8", bal), ("config3_fp8", "config3_fp8", bal),
             ("config2_append", "config2_append", bal), ("config3_append", "config3_append", bal),
             ("config2_fp8_append", "config2_fp8_append", bal)]
    runner, cur = None, None
    for key, name, pol in cases:
        try:
            if cur != name:
                runner = None
                torch.cuda.empty_cache()
                w = make_workload(name, args.seed)
                sms = torch.cuda.get_device_properties(device).multi_processor_count
                auto = default_policy(pkv, name, args, w, sms)
                runner = Runner(pkv, torch, w, pol or auto, rotation(torch, w, args, device), args.seed, device)
                cur = name
            pol = pol or auto
            w = runner.w
            K = w.steps if w.steps > 0 else 2 * args.graph_steps      # config 2 has no trace: 200 replayed steps
            chunk = max(1, min(args.graph_steps, K))
            bucketed = "buckets" in key
            whole_only = bucketed or runner.append is not None       # no decode-alone variant of these steps
            runner.set_bucket_route(1 if bucketed else None)
            r = time_policy(pkv, runner, pol, K, chunk, 5, decode_only=not whole_only)
            st = summarize(r["step_ms"], K)
            dc = summarize(r["decode_ms"], K) if not whole_only else st
            alg = mean_alg_bytes(w, K, runner.nlens)
            rows = pick_rows(runner.lens_at(0), 70000, w.seed)
            par, _ = parity_of(torch, runner, rows)
            c = runner.counters()      # after a whole eager step
            if bucketed:               # Table 4's counters of the bucket route, summed over the buckets
                hb = pkv.pkv_bucket_counters_host(runner.shape, pol, runner.lens_at(0), 1)
                c = dict(c, tasks=hb["tasks"], empty_tasks=hb["empty_tasks"], launched_build=0,
                         launched_decode=hb["decode_launches"], launched_merge=hb["merge_launches"])
            out[key] = {"workload": w.name, "policy": {k: int(v) for k, v in pol.__dict__.items()},
                        "steps": K, "us_per_step": round(st["us_per_step_median"], 3),
                        "us_per_step_min": round(st["us_per_step_min"], 3), "regions": st["regions"],
                        "decode_us": round(dc["us_per_step_median"], 3),
                        "alg_MB_per_step": round(alg / 1e6, 2),
                        "step_GBps": round(alg / st["us_per_step_median"] / 1e3, 1),
                        "decode_GBps": round(alg / dc["us_per_step_median"] / 1e3, 1),
                        "decode_frac_of_copy_peak": round(alg / dc["us_per_step_median"] / 1e3 / peak, 4),
                        "decode_frac_of_read_probe": round(alg / dc["us_per_step_median"] / 1e3 / read_peak, 4) if read_peak else None,
                        "decode_frac_of_8TBps": round(alg / dc["us_per_step_median"] / 1e3 / 8000.0, 4),
                        "tasks": c["tasks"], "empty_tasks": c["empty_tasks"],
                        "launches_per_step": c["launched_build"] + c["launched_decode"] + c["launched_merge"],
                        "parity": par}
            if key in ("config3", "config2_fp8") and not args.no_e2e:
                # the host-buffer step of these workloads too: pipelined and synchronous call, 200 steps each
                try:
                    es = run_e2e(pkv, torch, runner, 200, 5, auto=True)
                    ep = run_e2e_pipelined(pkv, torch, runner, 200, 5, auto=True)
                    out[key]["e2e"] = {"us_per_step": round(1e6 * ep[0] / 200, 2), "steps_enqueued_a_call_early": ep[2],
                                       "synchronous_us_per_step": round(1e6 * es[0] / 200, 2),
                                       "h2d_bytes_per_step": ep[1]["h2d_bytes"], "d2h_bytes_per_step": ep[1]["d2h_bytes"]}
                except Exception as ex:
                    out[key]["e2e"] = {"error": "%s: %s" % (type(ex).__name__, str(ex)[:200])}
        except Exception as e:      # an out-of-memory pool must not lose the headline line
            out[key] = {"error": "%s: %s" % (type(e).__name__, str(e)[:200])}
    runner = None
    torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------ launcher

def free_port():
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def relaunch_under_torchrun(args, argv):
    """`python bench.py --gpus N` (N > 1) outside torchrun: start N ranks of this same command."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "WARN")
    return subprocess.call(cmd, env=env)


def launcher_check(args):
    """The multi-rank plumbing without a GPU (gloo): rendezvous, barrier, MAX-over-ranks timing,
    whole-job aggregate, one JSON line from rank 0.  tests/test_multirank.py runs `--gpus 2` of it."""
    import torch.distributed as dist
    from paper_2606_26666_b200 import multirank
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    assert world == args.gpus, "WORLD_SIZE=%d but --gpus %d" % (world, args.gpus)
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    w = make_workload(args.workload, multirank.rank_seed(args.seed, rank), args.hkv)
    ms = 1.0 + rank                                         # stand-in device time of this rank
    ms_max, = multirank.max_over_ranks([ms])
    rows_all, = multirank.sum_over_ranks([w.B])
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"launcher_check": True, "n_gpus": world, "ms_max": ms_max, "rows_all": rows_all,
                          "value": multirank.whole_job_tokens_per_s(rows_all, args.steps, ms_max)}))
    return 0


# ------------------------------------------------------------------ the GPU arm

def sweep_on_tune_seed(pkv, torch, args, device, base_pol, K, W):
    """BASELINE.json configs[1]: split counts {1, 4, 16, 64} (FIXED_COUNT, 32-token tiles), plus the
    paper's auto rule (A12), a single-wave fit and the library's BALANCED policy -- timed on the
    TUNE seed 20260622, printed as information.  Returns (table, best policy)."""
    w = make_workload(args.workload, pkv_inputs.TUNE_SEED, args.hkv)
    runner = Runner(pkv, torch, w, base_pol, rotation(torch, w, args, device), pkv_inputs.TUNE_SEED, device)
    sms = torch.cuda.get_device_properties(device).multi_processor_count
    fixed = lambda S: dataclasses.replace(base_pol, tile_tokens=32, split_mode=pkv.SPLIT_FIXED_COUNT, num_splits=S)
    auto_pol = default_policy(pkv, args.workload, args, w, sms)
    cands = [(str(S), fixed(S)) for S in (1, 4, 16, 64, 0)] + [
        ("balanced", dataclasses.replace(base_pol, tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0)),
        ("cost_model", auto_pol)]
    s_fit = sms // max(1, w.B * w.Hkv)
    if s_fit > 1 and s_fit not in (4, 16, 64):
        cands.append((str(s_fit), fixed(s_fit)))
    Ks = min(K, 2 * args.graph_steps)
    chunk = max(1, min(args.graph_steps, Ks))
    table, pols = {}, {}
    for key, p2 in cands:
        r = time_policy(pkv, runner, p2, Ks, chunk, min(W, 5), decode_only=False)
        st = summarize(r["step_ms"], Ks)
        if key == "0":
            key = "auto(%d)" % r["counters"]["num_splits"]
        table[key] = {"us_per_step": round(st["us_per_step_median"], 3), "us_min": round(st["us_per_step_min"], 3),
                      "tasks": r["counters"]["tasks"],
                      "alg_GBps": round(algorithmic_bytes(w, w.seq_lens) / st["us_per_step_median"] / 1e3, 1)}
        pols[key] = p2
    best = min(table, key=lambda k_: table[k_]["us_per_step"])
    table["cost_model"]["policy"] = {k: int(v) for k, v in auto_pol.__dict__.items()}
    table["cost_model"]["vs_best_swept"] = round(table["cost_model"]["us_per_step"] / table[best]["us_per_step"], 4)
    del runner
    torch.cuda.empty_cache()
    return table, best, pols[best]


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2606_26666_b200 as pkv   # raises if libpkv.so is missing: there is no fallback
    from paper_2606_26666_b200 import multirank

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert world == args.gpus, "WORLD_SIZE=%d but --gpus %d: launch N ranks for --gpus N" % (world, args.gpus)
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    K, W = args.steps, max(args.warmup, 3)
    peak, peak_src = measured_hbm_peak()

    # beta / lambda of this device: the read-only streaming probe next to the copy peak
    cal = None
    try:
        if args.no_calibrate:
            raise RuntimeError("skipped (--no-calibrate)")
        buf = torch.empty(1 << 30, dtype=torch.uint8, device=device)
        cal = pkv.pkv_calibrate(buf)
        del buf
        torch.cuda.empty_cache()
    except Exception as e:
        cal = {"error": str(e)[:200]}
    read_peak = float(cal.get("read_gbps", 0.0)) if isinstance(cal, dict) else 0.0

    # every rank is a replica with its own seeded trace (data-parallel by row; DESIGN.md multi-GPU)
    seed = multirank.rank_seed(args.seed, rank)
    w = make_workload(args.workload, seed, args.hkv)
    sms = torch.cuda.get_device_properties(device).multi_processor_count
    pol = default_policy(pkv, args.workload, args, w, sms)
    chosen = "pkv_choose_policy (cost model, default B200 constants) on the step-0 lengths; no sweep involved"
    if args.split_mode >= 0 or args.splits >= 0 or args.tile_tokens > 0 or args.workload == "config1":
        chosen = "command line / BASELINE.json configs[0]"

    sweep = {}
    if args.workload == "config2" and not args.no_sweep and args.splits < 0:
        # information only: the timed policy is the cost model's, not the sweep's winner
        sweep, best_key, _ = sweep_on_tune_seed(pkv, torch, args, device, pol, K, W)
        sweep["fastest_on_tune_seed"] = best_key

    R = rotation(torch, w, args, device)
    runner = Runner(pkv, torch, w, pol, R, seed, device)
    chunk = max(1, min(args.graph_steps, K))
    counters = warm(pkv, runner, chunk, W)
    dec = pkv.STAGE_BUILD | pkv.STAGE_DECODE         # the decode kernel as the step launches it (fused build)
    runner.run(chunk, chunk, dec)                    # capture + warm the decode-only graphs too
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(device)
    sampler = ClockSampler(physical_gpu_index(local))
    sampler.start()
    step_ms = runner.run_repeated(K, chunk, pkv.STAGE_ALL)
    torch.cuda.synchronize(device)
    if world > 1:
        dist.barrier()
    dec_ms = runner.run_repeated(K, chunk, dec)
    clocks = sampler.result()

    e2e = e2e_pipe = None
    if not args.no_e2e:
        Ke = max(K, 200)      # a wall-clock number: at least 200 synchronised steps, however short the timed region K is
        e2e = run_e2e(pkv, torch, runner, Ke, W, auto=chosen.startswith("pkv_choose_policy"))
        try:
            e2e_pipe = run_e2e_pipelined(pkv, torch, runner, Ke, W, auto=chosen.startswith("pkv_choose_policy"))
        except Exception as ex:       # the synchronous call's number stands
            e2e_pipe = None
            sys.stderr.write("pipelined e2e skipped: %s\n" % str(ex)[:200])

    st, dc = summarize(step_ms, K), summarize(dec_ms, K)
    # max over ranks of the median region (and of the fastest one)
    # (a rank whose pipelined run was skipped counts with its synchronous time)
    ms_med, ms_min, ms_dec, e2e_s, e2e_pipe_s = multirank.max_over_ranks(
        [st["us_per_step_median"] * K / 1e3, st["us_per_step_min"] * K / 1e3, dc["us_per_step_median"] * K / 1e3,
         e2e[0] if e2e else 0.0, e2e_pipe[0] if e2e_pipe else (e2e[0] if e2e else 0.0)], device)
    rows_all, = multirank.sum_over_ranks([w.B], device)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    alg = mean_alg_bytes(w, K, runner.nlens)
    us_step, us_dec = 1e3 * ms_med / K, 1e3 * ms_dec / K
    launches_per_step = counters["launched_build"] + counters["launched_decode"] + counters["launched_merge"]
    cfg = workload_config(w, pol, R, args, world)
    cfg["policy_choice"] = chosen
    cfg["timing"] = {"regions_of_K_steps": st["regions"], "timed_ms_total": round(st["timed_ms_total"], 2),
                     "value_from": "median region",
                     "method": "region 1 between two synchronizes; the others back to back, each between two CUDA events on "
                               "the launching stream, one synchronize after the last",
                     "us_per_step_first_region": 1e3 * step_ms[0] / K, "us_per_step_median": st["us_per_step_median"],
                     "us_per_step_min": st["us_per_step_min"], "us_per_step_max": st["us_per_step_max"]}
    line = {
        "metric": "decode tokens/s", "value": multirank.whole_job_tokens_per_s(rows_all, K, ms_med), "unit": "tokens/s",
        "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_med / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f16", "data": "synthetic",
        "config": cfg,
        "us_per_step": us_step, "us_per_step_min": 1e3 * ms_min / K,
        "hbm_GBps_whole_step": alg / us_step / 1e3,
        "hbm_frac_whole_step": alg / us_step / 1e3 / peak,
        "hbm_frac_whole_step_of_8TBps": alg / us_step / 1e3 / 8000.0,
        "launches_per_step": {"build": counters["launched_build"], "decode": counters["launched_decode"],
                              "merge": counters["launched_merge"], "scheduler_decode": counters["decode_launches"],
                              "scheduler_merge": counters["merge_launches"], "tasks": counters["tasks"],
                              "num_splits": counters["num_splits"], "chunk_tiles": counters["chunk_tiles"],
                              "max_row_splits": counters["max_row_splits"]},
        "gpu_launches": int(launches_per_step * K * st["regions"]),
        "clocks": clocks,
        "calibration": cal,
        "roofline": {"bound": "hbm", "kernel": "pkv_decode_tma_kernel" if pol.kernel != pkv.KERNEL_SIMT else "pkv_decode_simt_kernel",
                     "achieved": alg / us_dec / 1e3, "peak": peak, "unit": "GB/s", "frac": alg / us_dec / 1e3 / peak,
                     "peak_source": peak_src, "frac_of_8TBps_nominal": alg / us_dec / 1e3 / 8000.0,
                     "read_probe_GBps": read_peak or None,
                     "frac_of_read_probe": (alg / us_dec / 1e3 / read_peak) if read_peak else None,
                     "algorithmic_bytes_per_launch": alg, "us_per_launch": us_dec,
                     "us_per_launch_min": dc["us_per_step_min"], "regions": dc["regions"], "traffic": None},
    }
    if sweep:
        line["config"]["split_sweep_tune_seed"] = sweep
    if e2e:
        c = e2e[1]
        line["e2e"] = {"value": rows_all * Ke / e2e_s, "unit": "tokens/s", "us_per_step": 1e6 * e2e_s / Ke, "steps": Ke,
                       "h2d_bytes_per_step": c["h2d_bytes"], "d2h_bytes_per_step": c["d2h_bytes"],
                       "api": "pkv_decode_host (host planning + H2D + launches + result in pinned host memory + sync per step)"}
        if e2e_pipe:
            # the serving loop's call (include/pkv.h pkv_decode_host_pipelined): the same bytes over the host link
            # and the same kernels per step, the next step's launches enqueued while this one runs
            cp = e2e_pipe[1]
            line["e2e"] = {"value": rows_all * Ke / e2e_pipe_s, "unit": "tokens/s", "us_per_step": 1e6 * e2e_pipe_s / Ke, "steps": Ke,
                           "h2d_bytes_per_step": cp["h2d_bytes"], "d2h_bytes_per_step": cp["d2h_bytes"],
                           "steps_enqueued_a_call_early": e2e_pipe[2],
                           "api": "pkv_decode_host_pipelined (each call is given the next step's lengths and table: host planning + "
                                  "launches of step t+1 during step t; per step q into pinned memory, flag, fetch over the host link, "
                                  "decode + merge, result in pinned host memory, done word)",
                           "synchronous": {"us_per_step": 1e6 * e2e_s / Ke, "value": rows_all * Ke / e2e_s,
                                           "api": "pkv_decode_host (host planning + H2D + launches + result in pinned host memory "
                                                  "+ sync per step)"}}

    # parity of the timed configuration + the oracle timed beside it (rank 0, N = 1)
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_of(torch, runner, args.cpu_seconds)
        line["parity"], _ = parity_of(torch, runner, pick_rows(runner.lens_at(0), 70000, w.seed))
    if args.timeline:
        write_timeline(torch, pkv, runner, args.timeline)
    if args.timeline_e2e:
        write_timeline_e2e(torch, pkv, runner, args.timeline_e2e, auto=chosen.startswith("pkv_choose_policy"))
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
    if world == 1 and not args.no_others and args.workload == "config2":
        del runner
        torch.cuda.empty_cache()
        line["config"]["other_workloads"] = other_workloads(pkv, torch, args, device, peak, read_peak)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    args = parse_args(argv)
    if args.impl == "reference" and not args.launcher_check:
        return run_reference(args)          # one process (rank 0 under torchrun), whatever --gpus says
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch_under_torchrun(args, argv)
    if args.launcher_check:
        return launcher_check(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
