"""N > 1 host logic on CPU: world_size-2 gloo processes shard a widened config-2
grid by rows dealt round-robin, integrate their shard (with the oracle here -- no GPU on this box) and the
scattered-back outputs equal the single-process result; the job time is the max over ranks.  bench.py's own
sharding path (global_workload / rank_shard) is driven for world sizes 2 and 8."""
import os
import socket

import numpy as np
import pytest

from paper_1802_00147_b200 import sharding, workloads

torch = pytest.importorskip("torch")


def test_scatter_back_inverts_the_round_robin_split():
    for rows, cols, world in [(3, 5, 2), (4, 7, 8), (1, 1, 3)]:
        glob = np.arange(rows * world * cols)
        parts = [glob[sharding.rank_orbits(rows, cols, r, world)] for r in range(world)]
        assert all(len(p) == rows * cols for p in parts)
        assert np.array_equal(sharding.scatter_back(parts, rows, cols, world), glob)
        two_d = [np.stack([p, -p]) for p in parts]
        assert np.array_equal(sharding.scatter_back(two_d, rows, cols, world), np.stack([glob, -glob]))


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
        q.put((rank, sharding.rank_rows(rows_per_rank, rank, world).tolist(), res.states, res.fli, res.status, job_ms, value))
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
    assert [g[1] for g in got] == [[0, 2, 4], [1, 3, 5]]                                # rows dealt round-robin
    back = lambda k: sharding.scatter_back([g[k] for g in got], rows_per_rank, cols, world)
    assert np.array_equal(back(2), ref.states)                                          # orbits are independent
    assert np.array_equal(back(3), ref.fli)
    assert np.array_equal(back(4), ref.status)
    assert all(g[5] == 20.0 for g in got)                                               # max over ranks
    expect = rows_per_rank * cols * n_steps * world / 20e-3
    assert all(abs(g[6] / expect - 1) < 1e-12 for g in got)


@pytest.mark.parametrize("world", [2, 8])
def test_bench_sharding_path_is_a_balanced_partition(world):
    """bench.py --gpus N: global_workload widens config 2 to 314 N rows over the same r0 range and rank_shard deals
    the rows round-robin.  The union of the shards is the N-wide grid, every rank holds 98 596 orbits, and every
    rank's r0 distribution spans [10, 60] with the same mean (within 1 %): no rank owns the strong-field band."""
    import argparse
    import bench
    args = argparse.Namespace(workload="config2", grid=314, n_steps=1000)
    full = bench.global_workload(args, world)
    assert full.n_orbits == 314 * 314 * world
    seen = np.zeros(full.n_orbits, dtype=int)
    means = []
    for rank in range(world):
        mine = bench.rank_shard(full, args, rank, world)
        assert mine.n_orbits == 314 * 314
        idx = sharding.rank_orbits(314, 314, rank, world)
        assert np.array_equal(mine.states, full.states[:, idx])
        seen[idx] += 1
        r0 = mine.states[0]
        assert r0.min() < 10.0 + 50.0 * world / (314 * world - 1) + 1e-9 and r0.max() > 60.0 - 50.0 * world / (314 * world - 1) - 1e-9
        means.append(r0.mean())
        strong = (r0 < 14.0).mean()                      # the band that holds every dropped cell
        assert abs(strong - 0.08) < 0.01
    assert (seen == 1).all()                              # disjoint and complete
    assert max(means) / min(means) - 1 < 0.01
    # a workload that is not the scan is replicated, not sharded
    args0 = argparse.Namespace(workload="config0", grid=314, n_steps=100)
    w0 = bench.global_workload(args0, world)
    assert bench.rank_shard(w0, args0, 1, world) is w0


@pytest.mark.parametrize("world", [2, 8])
def test_bench_strong_scaling_path_deals_the_same_grid(world):
    """bench.py --gpus N --scaling strong: the SAME 314 x 314 scan, row i on rank i mod N (n/G orbits per GPU).
    The shards are disjoint, complete, differ by at most one row, and every rank sees the whole r0 range."""
    import argparse
    import bench
    args = argparse.Namespace(workload="config2", grid=314, n_steps=1000, scaling="strong")
    full = bench.global_workload(args, world)
    assert full.n_orbits == 314 * 314
    seen = np.zeros(full.n_orbits, dtype=int)
    sizes = []
    for rank in range(world):
        mine = bench.rank_shard(full, args, rank, world)
        idx = sharding.strong_orbits(314, 314, rank, world)
        assert np.array_equal(mine.states, full.states[:, idx])
        seen[idx] += 1
        sizes.append(mine.n_orbits)
        r0 = mine.states[0]
        assert r0.min() < 10.0 + 50.0 * world / 313 + 1e-9 and r0.max() > 60.0 - 50.0 * world / 313 - 1e-9
    assert (seen == 1).all()
    assert max(sizes) - min(sizes) <= 314 and sum(sizes) == 314 * 314
    if world == 8:
        assert sorted(set(sizes)) == [39 * 314, 40 * 314]      # 12 246 / 12 560 orbits per rank
