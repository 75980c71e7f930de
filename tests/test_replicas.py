"""N > 1 host logic: the path shards as independent replicas, so the only cross-rank
steps are bookkeeping.  Covered here on CPU with the gloo backend, world_size 2."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2602_07397_b200.replicas import max_over_ranks, rank_seed, whole_job_throughput
    from synth import gen
    # every rank generates its own replica of a (tiny) planted layer from its own seed
    seed = rank_seed(2000, rank)
    q, k, v = gen.planted_qkv(seed, 256, 4, 2, 64, 64, torch.float32, [1, 2], [0, 1], device="cpu")
    digest = float(q.double().sum() + k.double().sum())
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms = max_over_ranks(ms_local, dist)
    gathered = [None] * world
    dist.all_gather_object(gathered, (seed, digest))
    dist.barrier()
    if rank == 0:
        out.put({"ms": ms, "value": whole_job_throughput(256 * 2, world, ms * 1e-3), "gathered": gathered})
    dist.destroy_process_group()


def test_two_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    res = out.get()
    assert res["ms"] == pytest.approx(15.0)            # max over ranks, not rank 0's own time
    assert res["value"] == pytest.approx(2 * 512 / 15e-3)
    (s0, d0), (s1, d1) = res["gathered"]
    assert s0 != s1 and d0 != d1                       # replicas hold different data


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    from paper_2602_07397_b200.replicas import max_over_ranks, rank_seed
    assert max_over_ranks(3.5) == 3.5
    assert rank_seed(7, 0) == 7
