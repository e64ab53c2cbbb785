"""N > 1 host logic on CPU: two gloo ranks, max-over-ranks timing and whole-job aggregation."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2004_02276_b200 import replicas
    local = 2.0 if rank == 0 else 4.0                   # rank 1 is the slow one
    dist.barrier()
    tmax = replicas.max_over_ranks(local)
    val = replicas.aggregate_throughput(1000, 10, local)
    q.put((rank, replicas.world(), tmax, val))
    dist.destroy_process_group()


def test_two_rank_aggregation():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, world, tmax, val in res:
        assert world == 2 and tmax == 4.0 and val == 2 * 1000 * 10 / 4.0


def test_single_process_identity():
    from paper_2004_02276_b200 import replicas
    assert replicas.world() == 1 and replicas.max_over_ranks(3.0) == 3.0
    assert replicas.aggregate_throughput(100, 2, 4.0) == 50.0
