"""world_size-2 gloo test of the N>1 host path (replicas only): chunk sharding covers every chunk
exactly once without communication, and the job time is the max over ranks."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_04410_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, ws, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    try:
        mine = replicas.shard_chunks(7, rank, ws)
        gathered = [None] * ws
        dist.all_gather_object(gathered, mine)
        ms = 10.0 + 5.0 * rank                        # rank 1 is slower
        total = replicas.max_over_ranks(ms)
        thr = replicas.job_throughput(8, 4, ms)
        q.put((rank, gathered, total, thr))
    finally:
        dist.destroy_process_group()


def test_replica_sharding_and_max_timing_gloo_ws2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = [q.get(timeout=120) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, gathered, total, thr in res:
        assert sorted(gathered[0] + gathered[1]) == list(range(7))          # every chunk exactly once
        assert not set(gathered[0]) & set(gathered[1])
        assert total == 15.0                                                 # max over ranks
        assert abs(thr - 2 * 8 * 4 / 15e-3) < 1e-6


def test_single_process_is_identity():
    assert replicas.world() == (0, 1)
    assert replicas.shard_chunks(3, 0, 1) == [0, 1, 2]
    assert replicas.max_over_ranks(3.5) == 3.5
