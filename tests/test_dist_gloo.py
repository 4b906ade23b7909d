"""World-size-2 gloo test of the N>1 host logic (timing reduction and event sharding); runs on CPU."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2505_22822_b200.dist import aggregate_throughput, shard_events


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank 0: 100 units in 10 ms; rank 1: 300 units in 20 ms  ->  400 units / 20 ms
    v, ms = aggregate_throughput(100.0 if rank == 0 else 300.0, 10.0 if rank == 0 else 20.0, 4, world)
    q.put((rank, v, ms, list(shard_events(7, rank, world))))
    dist.destroy_process_group()


def test_aggregate_is_sum_of_units_over_max_time():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
    for rank, v, ms, _ in res:
        assert abs(v - 400.0 / 0.020) < 1e-6
        assert abs(ms - 5.0) < 1e-9
    assert res[0][3] + res[1][3] == list(range(7))


def test_single_rank_passthrough():
    v, ms = aggregate_throughput(50.0, 25.0, 5, 1)
    assert v == 2000.0 and ms == 5.0
