"""N > 1 bookkeeping on CPU: world_size-2 `gloo` processes.

The path shards by row with no data-path collective, so what the ranks share is: the row split,
the per-rank seeded traces, the MAX-over-ranks timing and the whole-job aggregate -- plus the
property that makes row sharding exact: with a row-local split policy a rank's workqueue (host
planner of libpkv, through the C ABI) is exactly its rows' part of the full batch's queue, as the
workqueue oracle builds it.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import paper_2606_26666_b200 as pkv
from paper_2606_26666_b200 import multirank
from oracle import workqueue_oracle as wq

LENS = [700, 0, 33, 16, 257, 1, 2000, 31, 64, 65, 40000]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lens = np.array(LENS, dtype=np.int32)
        lo, hi = multirank.shard_rows(len(lens), world, rank)
        pol = pkv.Policy(tile_tokens=32, num_splits=5)
        shape = pkv.Shape(B=hi - lo, Hq=32, Hkv=8, max_pages=1, num_pages=1)
        tasks, offs = pkv.pkv_build_workqueue_host(shape, pol, lens[lo:hi])
        # the full queue from the oracle, restricted to this rank's rows and renumbered
        full = wq.build_workqueue(LENS, 8, wq.Policy(tile_tokens=32, num_splits=5))
        mine = [(r - lo, g, s, tb, te) for (r, g, s, tb, te) in full.tasks if lo <= r < hi]
        assert tasks.tolist() == [list(t) for t in mine]
        assert offs.tolist() == [o - full.split_offsets[lo] for o in full.split_offsets[lo:hi + 1]]
        # whole-job bookkeeping
        total_tasks, total_rows = multirank.sum_over_ranks([len(tasks), hi - lo])
        assert total_tasks == full.num_tasks and total_rows == len(LENS)
        ms_max, = multirank.max_over_ranks([10.0 + 5.0 * rank])
        assert ms_max == 10.0 + 5.0 * (world - 1)
        dist.barrier()
        seeds = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(seeds, torch.tensor([multirank.rank_seed(20260623, rank)]))
        assert [int(s) for s in seeds] == [20260623 + r for r in range(world)]
        ret[rank] = (lo, hi, multirank.whole_job_tokens_per_s(total_rows, 100, ms_max))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_row_sharding_and_timing():
    world = 2
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), ret), nprocs=world, join=True)
    assert sorted(ret.keys()) == [0, 1]
    (lo0, hi0, v0), (lo1, hi1, v1) = ret[0], ret[1]
    assert (lo0, hi1) == (0, len(LENS)) and hi0 == lo1          # a partition of the rows
    assert v0 == v1 == pytest.approx(len(LENS) * 100 / 15e-3)   # rows * steps / slowest rank


def test_shard_rows_partitions_exactly():
    for B in (0, 1, 7, 8, 128, 1001):
        for world in (1, 2, 3, 8):
            cuts = [multirank.shard_rows(B, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == B
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        multirank.shard_rows(8, 2, 2)


def test_single_process_reductions_are_identity():
    assert multirank.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert multirank.sum_over_ranks([3, 4]) == [3, 4]


def test_bench_gpus_2_spawns_two_ranks():
    """`python bench.py --gpus 2` outside torchrun must start two ranks itself (VERDICT r1 / ADVICE
    r1: the driver calls it exactly like this).  --launcher-check runs only the multi-rank
    plumbing (gloo rendezvous on 127.0.0.1, barrier, MAX over ranks, whole-job aggregate)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launcher-check", "--steps", "10",
                        "--workload", "config3"], capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["rows_all"] == 16          # two replicas of the B = 8 trace
    assert line["ms_max"] == 2.0                                    # MAX over ranks of (1.0, 2.0)
    assert line["value"] == 16 * 10 / 2.0e-3
