"""Multi-GPU host logic on CPU (world_size 2, gloo): the batch is sharded by configuration index with no data-path
collective (configurations are independent), timing is the max over ranks, the value is the whole-job sum."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        shard = bench.shard_batch(2, 6, rank)
        gathered = [None] * world
        dist.all_gather_object(gathered, (shard.offset, shard.symbol, shard.tau))
        ms = bench.reduce_max([10.0 + rank, 3.0 - rank], dist, "cpu")
        if rank == 0:
            q.put((gathered, ms))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_max_timing():
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    import bench
    from workloads import make_batch
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    gathered, ms = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    whole = make_batch(2, 12)
    sym = np.concatenate([g[1] for g in gathered])
    tau = np.concatenate([g[2] for g in gathered])
    lens = np.concatenate([np.diff(g[0]) for g in gathered])
    assert np.array_equal(sym, whole.symbol) and np.array_equal(tau, whole.tau)      # disjoint, ordered, complete
    assert np.array_equal(lens, np.diff(whole.offset))
    assert ms == [11.0, 3.0]                                                          # max over ranks
    assert bench.aggregate_value(2, 6, 5, 1000.0) == pytest.approx(60.0)             # whole-job traces/s


def test_reference_arm_runs_on_rank0_only(capsys):
    sys.path.insert(0, ROOT)
    import argparse
    import json
    import bench
    args = argparse.Namespace(config=1, steps=1, warmup=0, gpus=2)
    bench.run_reference(args, rank=1)
    assert capsys.readouterr().out == ""
    bench.REF_SAMPLE[1], keep = 32, bench.REF_SAMPLE[1]
    try:
        bench.run_reference(args, rank=0)
    finally:
        bench.REF_SAMPLE[1] = keep
    line = json.loads(capsys.readouterr().out)
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"
