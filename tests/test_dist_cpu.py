"""world_size-2 gloo tests (CPU) of the multi-process plumbing bench.py uses at N > 1: rendezvous on 127.0.0.1,
barrier, max-over-ranks timing and whole-job throughput."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    from paper_2605_09329_b200 import dist_util as D
    r, w = D.init("gloo")
    assert (r, w) == (rank, world)
    D.barrier()
    t_max = D.max_over_ranks(1.0 + rank)                 # rank 1 is the slow one
    total = D.sum_over_ranks(10.0)
    thr = D.job_throughput(30.0, 1.0 + rank)             # 30 steps per rank, 1 s and 2 s
    D.barrier()
    q.put((rank, t_max, total, thr))
    dist.destroy_process_group()


def test_two_rank_timing_reductions():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t_max, total, thr in out:
        assert t_max == 2.0 and total == 20.0
        assert thr == pytest.approx(60.0 / 2.0)          # all ranks' units over the slowest rank's time


def test_single_process_is_a_no_op():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_2605_09329_b200 import dist_util as D
    assert D.env_ranks() == (0, 1, 0)
    assert D.init("gloo") == (0, 1)
    assert D.max_over_ranks(3.5) == 3.5 and D.job_throughput(7.0, 2.0) == 3.5
