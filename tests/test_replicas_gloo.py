"""N > 1: `bench.py --gpus N` runs N independent replicas.  The only cross-rank logic is the
clock (max over ranks) and the whole-job value; covered here with world_size-2 gloo process groups on CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2501_02317_b200 import replicas


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local = 0.010 * (rank + 1)                      # rank 1 is the slow replica
        t = replicas.job_time(local)
        value, seconds = replicas.job_value(1000, 20, local)
        out.put((rank, t, value, seconds))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_job_time_is_max_over_ranks_and_value_is_whole_job():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, value, seconds in res:
        assert t == pytest.approx(0.020)                # the slow rank's time, on every rank
        assert seconds == pytest.approx(0.020)
        assert value == pytest.approx(1000 * 2 * 20 / 0.020)   # both replicas' work over the job time


def test_single_process_needs_no_process_group():
    assert replicas.job_time(0.5) == 0.5
    value, seconds = replicas.job_value(10, 3, 0.5)
    assert seconds == 0.5 and value == pytest.approx(60.0)
