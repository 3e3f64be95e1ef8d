"""N > 1 host logic on CPU: two gloo ranks shard the load cases and agree on the max-over-ranks time."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2410_20441_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lc = shard.load_case_of_rank(rank, world, base=2)
    ms = shard.max_over_ranks(10.0 + 5.0 * rank, dist)          # rank 1 is slower
    dist.barrier()
    out.put((rank, lc, ms))
    dist.destroy_process_group()


def test_two_ranks_shard_load_cases_and_take_max_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [2, 3]                         # distinct load cases
    assert all(g[2] == 15.0 for g in got)                        # max over ranks everywhere
    assert shard.job_throughput(1000, 10, world, 15.0) == pytest.approx(2 * 1000 * 10 / 0.015)


def test_single_process_paths():
    assert shard.load_case_of_rank(0, 1, base=2) == 2
    assert [shard.load_case_of_rank(r, 8, base=2) for r in range(8)] == [2, 3, 4, 5, 0, 1, 2, 3]
    assert shard.max_over_ranks(3.5, None) == 3.5
    with pytest.raises(ValueError):
        shard.load_case_of_rank(2, 2)
