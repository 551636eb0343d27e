"""N > 1 path of bench.py on CPU: two gloo ranks (127.0.0.1), no GPU.

The path shards by independent quartets: every rank draws its own seeded batch of the same
shape, there is no data-path collective, and the only exchange is the max-over-ranks of the step time.  This
covers that host logic: per-rank workloads, the MAX reduction and the whole-job rate.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = bench.workload_by_name("cfg2", rank)
        # every rank: same class and batch shape (weak scaling), its own seed and geometry
        fake_ms = 10.0 + 5.0 * rank           # rank 1 is the slow one
        ms = bench.reduce_max(fake_ms, world, "cpu")
        rate = bench.whole_job_rate(world, wl.nquartets, ms)
        digest = float(np.asarray(wl.shells.centers).sum())
        gathered = [None] * world
        dist.all_gather_object(gathered, (wl.seed, wl.nquartets, tuple(wl.lclass), digest))
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([ms, rate]))
        if rank == 0:
            import json
            json.dump(gathered, open(os.path.join(out_dir, "gathered.json"), "w"))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_by_independent_batches(tmp_path):
    world = 2
    mp.start_processes(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True, start_method="spawn")
    import json

    g = json.load(open(tmp_path / "gathered.json"))
    assert len(g) == world
    (s0, n0, c0, d0), (s1, n1, c1, d1) = g
    assert n0 == n1 == 4096 and c0 == c1 == [5, 5, 5, 5]      # same shape on every rank
    assert s0 != s1 and d0 != d1                              # different seeded shells
    for r in range(world):
        ms, rate = np.load(tmp_path / f"r{r}.npy")
        assert ms == 15.0                                     # max over ranks, seen by every rank
        assert rate == pytest.approx(world * 4096 / 15.0e-3)  # whole-job aggregate


def test_single_rank_helpers_need_no_process_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.reduce_max(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_rate(1, 16384, 65.0) == pytest.approx(16384 / 0.065)
