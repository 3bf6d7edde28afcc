"""World-size-2 gloo test (CPU) of bench.py's N > 1 host logic: replicas only, so
the only cross-rank step is the max-over-ranks timing and the whole-job rate built from it."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cpu")
    local_s = 0.010 * (rank + 1)                      # rank 1 is the slow one
    t = bench.max_over_ranks(local_s, dist, dev)
    v = bench.whole_job_rate(1000, 5, local_s, world, dist, dev)
    dist.barrier()
    out.put((rank, t, v))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate():
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
    for rank, t, v in res:
        assert t == pytest.approx(0.020)              # both ranks see the slowest rank's time
        assert v == pytest.approx(2 * 1000 * 5 / 0.020)


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.5, None, None) == 1.5
    assert bench.whole_job_rate(10, 2, 0.5, 1, None, None) == 40.0
