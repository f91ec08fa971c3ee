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


# ---- particle-sharded mode: partition logic and the row exchange, world_size 2 over gloo ----
def _row_from_fitness(rho_all, pst, r, lo, cnt):
    """What one rank contributes to an iteration, from the ORACLE's fitness values of its slice (the CUDA kernels cannot run
    here): sum w, sum w rho, sum w delta[6], |APS|, -, best exponent, best global index, its count, rho_ref, |O|, -."""
    import numpy as np
    rho_ref = rho_all[0]
    row = np.zeros(16)
    best_x, best_i = -np.log(rho_all[0]), 0
    for j in range(lo, lo + cnt):
        rj = rho_all[1 + j]
        if rj > rho_ref:
            w = rj - rho_ref
            row[0] += w; row[1] += w * rj; row[8] += 1
            row[2:8] += w * (r * pst[j].astype(np.float64))
        x = -np.log(rj)
        if x < best_x:
            best_x, best_i = x, 1 + j
    row[10], row[11], row[13] = best_x, best_i, rho_ref
    return row


def _shard_worker(rank, world, port, out):
    import numpy as np
    import oracle as orc
    import rf_synth as S
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N = 301
    pst = S.sample_pst(N, 77)
    rng = np.random.default_rng(5)
    rho_all = rng.uniform(0.3, 0.9, N + 1)
    r = np.array([0.02, 0.03, 0.04, 0.05, 0.06, 0.07])
    lo, cnt = replicas.particle_slices(N, world)[rank]
    row = torch.from_numpy(_row_from_fitness(rho_all, pst, r, lo, cnt))
    rows = torch.empty(world * 16, dtype=torch.float64)
    dist.all_gather_into_tensor(rows, row)                           # the ONE exchange of an iteration
    rows = rows.view(world, 16).numpy()
    sw, swr, sd, n_aps = rows[:, 0].sum(), rows[:, 1].sum(), rows[:, 2:8].sum(0), int(rows[:, 8].sum())
    b = min(range(world), key=lambda q: (rows[q, 10], rows[q, 11]))
    T = np.concatenate([np.eye(3), np.zeros((3, 1))], 1)
    want = orc.swarm_update(rho_all, pst, T, r)
    ok = (n_aps == want.n_aps and abs(sw - want.sum_omega) < 1e-12 and abs(swr / sw - want.rho_tilde) < 1e-12
          and np.allclose(sd / sw, list(want.delta_star), atol=1e-14) and int(rows[b, 11]) == want.argmax)
    out.put((rank, bool(ok), lo, cnt))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_particle_shards_fold_to_the_unsharded_update():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _, _ in got)
    assert got[0][2] == 0 and got[0][3] == 151 and got[1][2] == 151 and got[1][3] == 150      # contiguous, balanced, complete


def test_particle_slices_cover_the_template():
    for n, w in ((1024, 1), (1024, 8), (10240, 3), (7, 7), (131072, 5)):
        sl = replicas.particle_slices(n, w)
        assert len(sl) == w and sl[0][0] == 0 and sum(c for _, c in sl) == n
        assert all(sl[i][0] + sl[i][1] == sl[i + 1][0] for i in range(w - 1))
        assert max(c for _, c in sl) - min(c for _, c in sl) <= 1
    with pytest.raises(ValueError):
        replicas.particle_slices(3, 4)
