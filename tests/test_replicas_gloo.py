"""World-size-2 CPU test (gloo) of the multi-GPU bookkeeping bench.py uses in "replicas only" mode."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1707_08900_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world_size, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world_size)
    try:
        assert replicas.world() == (rank, world_size)
        replicas.barrier()
        ms = 10.0 + 5.0 * rank  # rank 1 is the slow one
        ms_max = replicas.max_over_ranks(ms)
        value = replicas.whole_job_value(1000, 4, ms_max, world_size)
        replicas.barrier()
        out.put((rank, ms_max, value))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world_size_2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # both ranks see the slow rank's time; value counts the cells of BOTH ranks over that time
    assert [g[1] for g in got] == [15.0, 15.0]
    expect = 2 * 1000 * 4 / 15.0e-3 / 1e6
    assert all(abs(g[2] - expect) < 1e-12 for g in got)


def test_single_process_defaults():
    assert replicas.world() == (0, 1)
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_value(8, 2, 4.0, 1) == pytest.approx(8 * 2 / 4.0e-3 / 1e6)
    with pytest.raises(ValueError):
        replicas.whole_job_value(8, 2, 0.0, 1)
