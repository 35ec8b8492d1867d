"""world_size-2 CPU test (gloo) of the N > 1 path's host logic: the session -> rank map is a
partition, replicas draw different inputs, and the timed region is reduced as max over ranks with
the whole-job throughput summed over ranks (the contract bench.py follows)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_02640_b200 import replicas, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = replicas.local_sessions(10, world, rank)
    ms_local = 2.0 + rank                      # rank 1 is the slow one
    value, ms = replicas.aggregate(ms_local, 100.0 * len(mine))
    dist.barrier()
    rows = synth.rows(1, synth.STREAM_K, 0, torch.tensor([replicas.uid_base(rank)]), torch.tensor([0]), 2, 64)
    q.put((rank, mine, value, ms, rows.float().sum().item()))
    dist.destroy_process_group()


def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, v0, ms0, x0), (r1, s1, v1, ms1, x1) = out
    assert sorted(s0 + s1) == list(range(10)) and not set(s0) & set(s1)        # a partition
    assert ms0 == ms1 == 3.0                                                    # max over ranks
    assert abs(v0 - 1000.0 / 3e-3) < 1e-6 and v0 == v1                          # whole-job aggregate
    assert x0 != x1                                                             # replicas are not clones


def test_single_process_aggregate_is_identity():
    value, ms = replicas.aggregate(4.0, 200.0)
    assert ms == 4.0 and abs(value - 200.0 / 4e-3) < 1e-9
