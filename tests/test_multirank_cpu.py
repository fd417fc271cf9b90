"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- no data-path collective;
the only exchange is the timing / work aggregation (max over ranks, sum over ranks)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms, upd = bench.aggregate(10.0 + 5.0 * rank, 1000 * (rank + 1), "cpu")
    q.put((rank, ms, upd))
    dist.destroy_process_group()


def test_aggregate_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, ms, upd in res:
        assert ms == 15.0          # max over ranks
        assert upd == 3000.0       # whole-job work = sum over ranks


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 7) == (3.5, 7)
