"""N > 1 host logic on CPU: world_size-2 gloo processes shard a widened config-2
grid by contiguous orbit ranges, integrate their shard (with the oracle here -- no GPU on this box) and
the concatenation equals the single-process result; the job time is the max over ranks."""
import os
import socket

import numpy as np
import pytest

from paper_1802_00147_b200 import sharding, workloads

torch = pytest.importorskip("torch")


def test_shard_ranges_partition_the_index_range():
    for n, world in [(314, 1), (314, 2), (628, 8), (7, 3), (2, 4), (0, 2)]:
        spans = [workloads.shard_range(n, r, world) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))            # contiguous, disjoint
        sizes = [hi - lo for lo, hi in spans]
        assert max(sizes) - min(sizes) <= 1                                   # balanced


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, rows_per_rank, cols, n_steps, q):
    import torch.distributed as dist
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        full = workloads.config2(n_r=rows_per_rank * world, n_theta=cols, n_steps=n_steps)
        mine = sharding.rank_shard(full, rows_per_rank, cols, rank, world)
        res = oracle.integrate(mine.states, mine.h, n_steps, 3, shadow_eps=mine.shadow_eps, n_threads=1, **mine.params())
        local_ms = 10.0 * (rank + 1)                                          # rank 1 is the slow one
        job_ms = sharding.max_over_ranks(local_ms)
        value = sharding.job_throughput(mine.n_orbits * n_steps, world, 1, local_ms)
        q.put((rank, sharding.rank_rows(rows_per_rank, rank, world), res.states, res.fli, res.status, job_ms, value))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_single_process_scan():
    import torch.multiprocessing as mp
    import oracle
    world, rows_per_rank, cols, n_steps = 2, 3, 5, 200
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, rows_per_rank, cols, n_steps, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=120) for _ in procs], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = workloads.config2(n_r=rows_per_rank * world, n_theta=cols, n_steps=n_steps)
    ref = oracle.integrate(full.states, full.h, n_steps, 3, shadow_eps=full.shadow_eps, n_threads=1, **full.params())
    assert [g[1] for g in got] == [(0, 3), (3, 6)]
    assert np.array_equal(np.concatenate([g[2] for g in got], axis=1), ref.states)     # orbits are independent
    assert np.array_equal(np.concatenate([g[3] for g in got]), ref.fli)
    assert np.array_equal(np.concatenate([g[4] for g in got]), ref.status)
    assert all(g[5] == 20.0 for g in got)                                               # max over ranks
    expect = rows_per_rank * cols * n_steps * world / 20e-3
    assert all(abs(g[6] / expect - 1) < 1e-12 for g in got)
