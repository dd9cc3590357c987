"""bench.py --gpus N runs N independent replicas.  The only multi-rank logic
is the barrier around the timed region, the max-over-ranks reduction of the device time and the whole-job rate:
covered here with two CPU processes over gloo."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp

from paper_2306_09855_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world), RANK=str(rank),
                      LOCAL_RANK=str(rank))
    assert replicas.env_world() == (world, rank, rank)
    dist = replicas.init("gloo")
    replicas.barrier(dist)
    ms = 10.0 + 5.0 * rank  # rank 1 is the slow replica
    slowest = replicas.max_over_ranks(dist, ms)
    rate = replicas.whole_job_rate(1000, 4, world, slowest)
    replicas.barrier(dist)
    out[rank] = (slowest, rate)
    dist.destroy_process_group()


def test_two_replicas_reduce_to_the_slowest_rank():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    slowest, rate = res[0]
    assert slowest == 15.0
    assert rate == pytest.approx(2 * 1000 * 4 / 15e-3)


def test_single_process_needs_no_process_group(monkeypatch):
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert replicas.env_world() == (1, 0, 0)
    assert replicas.init("gloo") is None
    assert replicas.max_over_ranks(None, 7.5) == 7.5
    assert replicas.whole_job_rate(100, 2, 1, 10.0) == pytest.approx(100 * 2 / 10e-3)
