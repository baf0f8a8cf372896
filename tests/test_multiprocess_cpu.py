"""The N > 1 timing plumbing of bench.py (the slab exchange itself is tests/test_slab_cpu.py) on CPU: two gloo ranks
rendezvous on 127.0.0.1, the per-rank times are max-reduced and the whole-job numbers follow."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 * (rank + 1)                    # rank 1 is the slow one
        dist.barrier()
        ms = bench.reduce_max(ms_local, world, "cpu")
        job = bench.job_numbers(ms, 1000, world)
        out.put((rank, ms, job["grind_ns"], job["cell_updates_per_s"]))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_max_reduce_and_job_metric():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, grind, cups in res:
        assert ms == 20.0                                   # max over ranks
        assert grind == pytest.approx(20.0 * 1e6 / (2000 * 15))
        assert cups == pytest.approx(2000 / 20e-3)          # aggregate over both ranks


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max(3.5, 1) == 3.5
    one, two = bench.job_numbers(10.0, 1000, 1), bench.job_numbers(10.0, 1000, 2)
    assert two["cell_updates_per_s"] == 2 * one["cell_updates_per_s"]     # weak scaling
    assert two["grind_ns"] == pytest.approx(one["grind_ns"] / 2)
