"""The N>1 path of bench.py (independent replicas; barrier + max-over-ranks timing + summed units) on the
CPU with the gloo backend, world_size 2."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2406_03243_b200 import replicas
    replicas.barrier()
    ms = replicas.max_over_ranks(1.0 + rank)              # rank 1 is the slow one
    units = replicas.sum_over_ranks(10.0 * (rank + 1))    # 10 + 20
    thr = replicas.aggregate_throughput(100.0, 2.0 + 2.0 * rank)
    out.put((rank, replicas.world_size(), ms, units, thr))
    dist.destroy_process_group()


def test_replica_aggregation_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, world, ms, units, thr in res:
        assert world == 2 and ms == 2.0 and units == 30.0 and thr == 200.0 / 4.0


def test_single_process_is_identity():
    from paper_2406_03243_b200 import replicas
    assert replicas.world_size() == 1
    assert replicas.max_over_ranks(3.5) == 3.5 and replicas.sum_over_ranks(2.0) == 2.0
    assert replicas.aggregate_throughput(8.0, 2.0) == 4.0
    replicas.barrier()
