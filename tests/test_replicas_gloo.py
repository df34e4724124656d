"""N > 1 plumbing on CPU: two gloo ranks run the reductions bench.py uses for replicas (max-over-ranks time,
whole-job throughput) and get distinct Philox keys.  The data path itself has no collective."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_15073_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = replicas.max_over_ranks(10.0 + 5.0 * rank, dist)                       # rank 1 is the slow one
    thr = replicas.aggregate_throughput(1000.0 * (rank + 1), 2.0 + rank, dist)  # 3000 units / max(2, 3) s
    out.put((rank, t, thr, replicas.rank_seed(3001, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_reductions_and_seeds():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]
    assert [r[2] for r in res] == [1000.0, 1000.0]
    assert res[0][3] == 3001 and res[1][3] != res[0][3] and 0 <= res[1][3] < 2 ** 64


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.aggregate_throughput(10.0, 4.0) == 2.5
    assert replicas.rank_seed(7, 0) == 7
