"""N>1 path of bench.py on CPU: two gloo ranks, max-over-ranks timing, whole-job aggregate (replicas only)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1307_6488_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local = 0.5 if rank == 0 else 2.0          # rank 1 is the slow replica
    value, worst = replicas.aggregate_throughput(local, 1000.0, dist)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, value, worst, replicas.replica_seed(100, rank)))


def test_two_rank_aggregate():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, worst, seed in res:
        assert worst == 2.0                    # max over ranks
        assert value == 2 * 1000.0 / 2.0       # whole job = all ranks' units / slowest time
        assert seed == 100 + rank


def test_single_process():
    value, worst = replicas.aggregate_throughput(0.25, 10.0)
    assert (value, worst) == (40.0, 0.25)
