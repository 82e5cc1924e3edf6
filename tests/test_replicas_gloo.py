"""world_size-2 gloo test (CPU) of the replica plumbing bench.py uses under torchrun: barrier, MAX over ranks of the
per-rank step time, whole-job aggregate.  The hot path itself never spans GPUs."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2607_03226_b200 import replicas
    assert replicas.env_rank() == (rank, world, rank)
    dist = replicas.init("gloo")
    replicas.barrier(dist)
    ms = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
    worst = replicas.max_over_ranks(ms, dist)
    rate = replicas.whole_job_rate(1000, world, worst * 1e-3)
    replicas.barrier(dist)
    out.put((rank, worst, rate))
    dist.destroy_process_group()


def test_two_replicas_time_as_the_slowest_and_add_up():
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
    for rank, worst, rate in res:
        assert worst == 15.0
        assert abs(rate - 2 * 1000 / 15e-3) < 1e-6


def test_single_process_needs_no_group():
    from paper_2607_03226_b200 import replicas
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.init("gloo") is None
    assert replicas.max_over_ranks(3.5, None) == 3.5
    replicas.barrier(None)
