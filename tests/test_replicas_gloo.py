"""N > 1 host logic on CPU: world_size-2 gloo run of the replicas-only aggregation used by bench.py --gpus N."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2105_05600_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, units = (10.0, 1000.0) if rank == 0 else (12.5, 900.0)
    t, u = replicas.aggregate(ms, units)
    out.put((rank, t, u, replicas.shard_start(rank, 53)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregate_is_max_time_and_sum_units():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, u, start in got:
        assert t == 12.5 and u == 1900.0            # max over ranks of the time, sum over ranks of the work
    assert got[0][3] != got[1][3]                   # each rank tracks its own stretch of the trajectory


def test_single_process_and_shard_bounds():
    assert replicas.aggregate(3.0, 7.0) == (3.0, 7.0)
    for n in (23, 53, 200):
        for r in range(8):
            s = replicas.shard_start(r, n)
            assert 0 <= s and s + n <= 200
    with pytest.raises(ValueError):
        replicas.shard_start(0, 201)
