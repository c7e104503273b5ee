"""pkv_decode_host_pipelined (include/pkv.h "The host-buffer step with its submission taken off the
critical path"): the next step's launches are enqueued behind a gate kernel while the current step
runs.  The kernels and their inputs are those of pkv_decode_host, so every step must equal the plain
call's result BIT FOR BIT -- through correct predictions, mispredictions (the armed step is discarded),
table changes, steps that arm nothing, and drains.  Parity of pkv_decode_host itself with the oracle is
test_gpu_parity.py's business.

While a step is armed the stream is blocked (for at most the gate's 200 ms), so nothing here touches
the device between pipelined calls except through the decoder, and every case ends drained -- but for
the one test that lets a gate expire on purpose."""
import time

import numpy as np
import pytest
import torch

import paper_2606_26666_b200 as pkv
from gpu_helpers import DevProblem
from helpers import make_problem

pytestmark = pytest.mark.gpu

STEPS = 24


class Loop:
    """A serving loop's host state: growing rows, one request replaced at step 5, one finished at step 9."""

    def __init__(self, pol, seed=2100, lens=(1500, 62, 4000, 333)):
        self.lens0 = np.array(lens, dtype=np.int32)
        self.p = p = make_problem(list(self.lens0 + STEPS + 8), seed=seed)
        p2 = make_problem(list(self.lens0 + STEPS + 8), seed=seed + 1)
        self.alt_row = p2.block_table[1] % p.k_cache.shape[0]
        self.dp = DevProblem(p)
        self.pol = pol
        self.stream = torch.cuda.Stream()
        rng = np.random.Generator(np.random.PCG64(seed))
        self.q = [torch.from_numpy(rng.standard_normal(p.q.shape).astype(np.float16)).pin_memory() for _ in range(3)]
        self.tables, self.lens = [], []
        table = p.block_table.copy()
        for t in range(STEPS + 1):
            cur = (self.lens0 + t).astype(np.int32)
            if t >= 5:
                table = table.copy()
                table[1] = self.alt_row
            if t >= 9:
                cur[3] = 0
            self.tables.append(torch.from_numpy(np.ascontiguousarray(table)).pin_memory())
            self.lens.append(torch.from_numpy(cur).pin_memory())
        self.out = torch.full((p.B, p.Hq, p.d), float("nan"), dtype=torch.float16).pin_memory()

    def buffers(self):
        nb = pkv.pkv_host_scratch_bytes(self.dp.shape, self.pol)
        return (torch.zeros(nb, dtype=torch.uint8).pin_memory(), torch.empty(nb, dtype=torch.uint8, device="cuda"),
                pkv.alloc_workspace(self.dp.shape, self.pol))

    def plain_pass(self):
        staging, scratch, ws = self.buffers()
        dec = pkv.HostDecoder(self.dp.shape, self.pol, self.dp.k, self.dp.v, staging, scratch, ws, self.p.scale, stream=self.stream)
        outs, counters = [], []
        for t in range(STEPS):
            self.out.fill_(float("nan"))
            dec(self.q[t % 3].data_ptr(), self.tables[t].data_ptr(), self.lens[t].data_ptr(), self.out.data_ptr())
            outs.append(self.out.numpy().copy())
            counters.append(dec.counters)
        return outs, counters


POLICIES = [pkv.Policy(tile_tokens=32, num_splits=5, flags=pkv.FLAG_OUT_PINNED),
            pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_BALANCED, num_splits=0, flags=pkv.FLAG_OUT_PINNED),
            pkv.Policy(tile_tokens=16, split_mode=pkv.SPLIT_AUTO, num_splits=0, flags=pkv.FLAG_OUT_PINNED),
            pkv.Policy(tile_tokens=32, num_splits=3, merge_mode=pkv.MERGE_FUSED)]


@pytest.mark.parametrize("pol", POLICIES, ids=["fixed5", "balanced", "auto", "fused3_uncached_ptrs"])
@pytest.mark.parametrize("predict", ["right", "sometimes_wrong", "never"])
def test_pipelined_steps_equal_the_plain_call_bit_for_bit(pol, predict):
    lp = Loop(pol)
    want, want_c = lp.plain_pass()
    assert not np.isnan(want[0]).any() and not np.array_equal(want[0], want[1])
    staging, scratch, ws = lp.buffers()
    dec = pkv.PipelinedHostDecoder(lp.dp.shape, pol, lp.dp.k, lp.dp.v, staging, scratch, ws, lp.p.scale, stream=lp.stream)
    wrong = lp.lens[0].clone()          # a prediction that never comes true
    wrong += 3
    armed = 0
    try:
        for t in range(STEPS):
            nl, nt = lp.lens[t + 1].data_ptr(), lp.tables[t + 1].data_ptr()
            if predict == "never":
                nl = nt = 0
            elif predict == "sometimes_wrong" and t % 4 == 2:
                nl = wrong.data_ptr()
            elif predict == "sometimes_wrong" and t % 4 == 3:
                nt = lp.tables[0].data_ptr() if t >= 5 else lp.tables[STEPS].data_ptr()      # the other table
            lp.out.fill_(float("nan"))
            dec(lp.q[t % 3].data_ptr(), lp.tables[t].data_ptr(), lp.lens[t].data_ptr(), lp.out.data_ptr(), nl, nt)
            assert np.array_equal(lp.out.numpy().view(np.uint16), want[t].view(np.uint16)), "step %d" % t
            c = dec.counters
            for key in ("tasks", "decode_launches", "merge_launches", "max_row_splits", "d2h_bytes"):
                assert c[key] == want_c[t][key], (t, key)
            armed += c["armed_step"]
    finally:
        dec.drain()
    torch.cuda.synchronize()            # returns: nothing is armed any more
    # the pipeline really is used: a correctly predicted step whose kernels have run before was enqueued a call early
    if predict == "never":
        assert armed == 0
    elif predict == "right":
        assert armed >= STEPS - 4, armed      # not the first step, nor the step after a change of the launch signature
    else:
        assert 0 < armed < STEPS - 4, armed


def test_plain_call_and_synchronize_after_an_armed_step():
    """pkv_decode_host on a staging buffer with an armed step drains it first; drain() is idempotent; a
    pageable out_host (no device mapping) makes the pipelined call fall back to the plain one."""
    pol = pkv.Policy(tile_tokens=32, num_splits=4, flags=pkv.FLAG_OUT_PINNED)
    lp = Loop(pol, seed=2200)
    want, _ = lp.plain_pass()
    staging, scratch, ws = lp.buffers()
    dec = pkv.PipelinedHostDecoder(lp.dp.shape, pol, lp.dp.k, lp.dp.v, staging, scratch, ws, lp.p.scale, stream=lp.stream)
    for t in range(3):
        dec(lp.q[t % 3].data_ptr(), lp.tables[t].data_ptr(), lp.lens[t].data_ptr(), lp.out.data_ptr(),
            lp.lens[t + 1].data_ptr(), lp.tables[t + 1].data_ptr())
        assert np.array_equal(lp.out.numpy().view(np.uint16), want[t].view(np.uint16))
    # step 3 is armed now; the plain entry point on the same buffers must not hang
    plain = pkv.HostDecoder(lp.dp.shape, pol, lp.dp.k, lp.dp.v, staging, scratch, ws, lp.p.scale, stream=lp.stream)
    plain(lp.q[0].data_ptr(), lp.tables[3].data_ptr(), lp.lens[3].data_ptr(), lp.out.data_ptr())
    assert np.array_equal(lp.out.numpy().view(np.uint16), want[3].view(np.uint16))
    dec.drain()
    dec.drain()
    torch.cuda.synchronize()
    # pageable out: falls back, same bits
    pageable = np.full(lp.out.shape, np.nan, dtype=np.float16)
    dec(lp.q[1].data_ptr(), lp.tables[4].data_ptr(), lp.lens[4].data_ptr(), pageable.ctypes.data, lp.lens[5].data_ptr(), lp.tables[5].data_ptr())
    assert np.array_equal(pageable.view(np.uint16), want[4].view(np.uint16))
    dec.drain()
    torch.cuda.synchronize()


def test_unreleased_step_expires_and_is_redone():
    """A device-wide synchronisation while a step is armed does not deadlock: the gate gives up after its
    timeout (200 ms), the step runs on stale inputs and is marked expired, and the next call -- which
    would have released it -- does the step again instead of trusting its result."""
    pol = pkv.Policy(tile_tokens=32, num_splits=4, flags=pkv.FLAG_OUT_PINNED)
    lp = Loop(pol, seed=2300)
    want, _ = lp.plain_pass()
    staging, scratch, ws = lp.buffers()
    dec = pkv.PipelinedHostDecoder(lp.dp.shape, pol, lp.dp.k, lp.dp.v, staging, scratch, ws, lp.p.scale, stream=lp.stream)
    for t in range(3):
        dec(lp.q[t % 3].data_ptr(), lp.tables[t].data_ptr(), lp.lens[t].data_ptr(), lp.out.data_ptr(),
            lp.lens[t + 1].data_ptr(), lp.tables[t + 1].data_ptr())
    assert dec.counters["armed_step"] == 1                    # step 2 had been armed by step 1's call; step 3 is armed now
    assert not lp.stream.query()                              # the gate of step 3 holds the stream
    t0 = time.perf_counter()
    torch.cuda.synchronize()                                  # no drain: waits for the gate to give up
    waited = time.perf_counter() - t0
    assert 0.05 < waited < 5.0, waited
    lp.out.fill_(float("nan"))
    dec(lp.q[0].data_ptr(), lp.tables[3].data_ptr(), lp.lens[3].data_ptr(), lp.out.data_ptr(), lp.lens[4].data_ptr(), lp.tables[4].data_ptr())
    assert np.array_equal(lp.out.numpy().view(np.uint16), want[3].view(np.uint16))
    assert dec.counters["armed_step"] == 0                    # redone, not released
    dec(lp.q[1].data_ptr(), lp.tables[4].data_ptr(), lp.lens[4].data_ptr(), lp.out.data_ptr())
    assert np.array_equal(lp.out.numpy().view(np.uint16), want[4].view(np.uint16))
    assert dec.counters["armed_step"] == 1                    # the pipeline is back in step
    dec.drain()
    torch.cuda.synchronize()


def test_prepared_calls_replay_the_same_step_arguments():
    """PipelinedHostDecoder.prepare() / run(): the marshalled argument list of a step, built once."""
    pol = pkv.Policy(tile_tokens=32, num_splits=4, flags=pkv.FLAG_OUT_PINNED)
    lp = Loop(pol, seed=2400)
    want, _ = lp.plain_pass()
    staging, scratch, ws = lp.buffers()
    dec = pkv.PipelinedHostDecoder(lp.dp.shape, pol, lp.dp.k, lp.dp.v, staging, scratch, ws, lp.p.scale, stream=lp.stream)
    steps = [dec.prepare(lp.q[t % 3].data_ptr(), lp.tables[t].data_ptr(), lp.lens[t].data_ptr(), lp.out.data_ptr(),
                         lp.lens[t + 1].data_ptr(), lp.tables[t + 1].data_ptr()) for t in range(8)]
    armed = 0
    try:
        for t in range(8):
            lp.out.fill_(float("nan"))
            dec.run(steps[t])
            assert np.array_equal(lp.out.numpy().view(np.uint16), want[t].view(np.uint16)), "step %d" % t
            armed += dec.counters["armed_step"]
    finally:
        dec.drain()
    assert armed >= 5
    torch.cuda.synchronize()


def test_pipelined_steps_on_fp8_caches():
    """The pipeline is the host path around the same launches: one-byte caches (per-head scales in the
    shape) go through it unchanged, bit-identical to the plain call."""
    from test_gpu_fp8 import Fp8Problem
    pol = pkv.Policy(tile_tokens=32, num_splits=5, flags=pkv.FLAG_OUT_PINNED)
    lp = Loop(pol, seed=2500)
    lp.dp = Fp8Problem(list(lp.lens0 + STEPS + 8), seed=2500)       # the same tables and pool size; E4M3 bytes, scales
    assert np.array_equal(lp.dp.p.block_table, lp.p.block_table) and lp.dp.shape.kv_dtype == pkv.KV_E4M3
    want, _ = lp.plain_pass()
    assert not np.isnan(want[0]).any()
    staging, scratch, ws = lp.buffers()
    dec = pkv.PipelinedHostDecoder(lp.dp.shape, pol, lp.dp.k, lp.dp.v, staging, scratch, ws, lp.p.scale, stream=lp.stream)
    armed = 0
    try:
        for t in range(STEPS):
            lp.out.fill_(float("nan"))
            dec(lp.q[t % 3].data_ptr(), lp.tables[t].data_ptr(), lp.lens[t].data_ptr(), lp.out.data_ptr(),
                lp.lens[t + 1].data_ptr(), lp.tables[t + 1].data_ptr())
            assert np.array_equal(lp.out.numpy().view(np.uint16), want[t].view(np.uint16)), "step %d" % t
            armed += dec.counters["armed_step"]
    finally:
        dec.drain()
    assert armed >= STEPS - 4
    torch.cuda.synchronize()
