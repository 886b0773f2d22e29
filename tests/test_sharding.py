"""Host logic of the multi-GPU path on CPU: id ranges are disjoint and cover the job; the
max-over-ranks / sum-over-ranks reduction works across two gloo processes; sharded oracle runs reproduce the
unsharded one (outputs are a function of (inputs, seed, id) only)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shards_partition_the_ids():
    from paper_2512_10520_b200.sharding import strong_shard, weak_shard
    for n_total, world in ((10, 3), (7, 8), (0, 2), (10_000_001, 8), (64, 1)):
        shards = [strong_shard(n_total, r, world) for r in range(world)]
        assert shards[0].id_base == 0 and sum(s.n for s in shards) == n_total
        for a, b in zip(shards, shards[1:]):
            assert a.id_base + a.n == b.id_base and a.n - b.n in (0, 1)
    w = [weak_shard(1000, r, 4) for r in range(4)]
    assert [s.id_base for s in w] == [0, 1000, 2000, 3000] and all(s.n == 1000 for s in w)
    with pytest.raises(ValueError):
        strong_shard(10, 3, 3)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle
    from paper_2512_10520_b200 import workloads as w
    from paper_2512_10520_b200.sharding import gather_ranges, reduce_job, strong_shard
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = w.config1(n=2001, n_draws=20_000)
        sh = strong_shard(len(wl.muons.pos_q), rank, world)
        sel = slice(sh.id_base, sh.id_base + sh.n)
        r = oracle.transport(oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom), wl.muons.pos_q[sel],
                             wl.muons.mom[sel], wl.seed, id_base=sh.id_base, threads=1)
        times, totals = reduce_job([0.5 + rank, 2.0 - rank], [int(r["steps"].sum()), sh.n], dist)
        np.savez(os.path.join(out_dir, "rank%d.npz" % rank), pos=r["pos"], mom=r["mom"], flag=r["flag"],
                 steps=r["steps"], id_base=sh.id_base, times=times, totals=totals, ranges=gather_ranges(sh, dist))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_job_equals_the_unsharded_one(tmp_path, oracle, workloads):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    wl = workloads.config1(n=2001, n_draws=20_000)
    ref = oracle.transport(oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom), wl.muons.pos_q,
                           wl.muons.mom, wl.seed, threads=1)
    parts = [np.load(os.path.join(tmp_path, "rank%d.npz" % r)) for r in range(world)]
    assert [int(p["id_base"]) for p in parts] == [0, 1001]
    for k in ("pos", "mom", "flag", "steps"):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), ref[k])
    for p in parts:                                   # every rank sees the id ranges all ranks report: disjoint, covering
        assert p["ranges"].tolist() == [[0, 1001], [1001, 2001]]
    for p in parts:                                   # every rank holds the same whole-job figures
        assert list(p["times"]) == [1.5, 2.0]        # max over ranks
        assert list(p["totals"]) == [float(ref["steps"].sum()), 2001.0]


# ------------------------------------------------------------- configs[4] across ranks: whole batches, k -> rank k % N
def test_batches_are_dealt_round_robin():
    from paper_2512_10520_b200.sharding import batch_shard
    for n_batches, world in ((10, 1), (10, 2), (10, 4), (10, 8), (3, 8), (0, 2)):
        dealt = [batch_shard(n_batches, r, world) for r in range(world)]
        assert sorted(k for d in dealt for k in d) == list(range(n_batches))          # each batch once
        assert max(len(d) for d in dealt) - min(len(d) for d in dealt) <= 1
        assert all(k % world == r for r, d in enumerate(dealt) for k in d)
    with pytest.raises(ValueError):
        batch_shard(10, 2, 2)


N_BATCH, BATCHES = 301, 4


def _batch_worker(rank, world, port, out_dir):
    """One rank of `bench.py --sweep --gpus N` with the oracle in the kernels' place: its batches, its ids, the job's
    reduction."""
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle
    from paper_2512_10520_b200 import workloads as w
    from paper_2512_10520_b200.sharding import batch_shard, reduce_job
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = w.config1(n=8, n_draws=20_000)
        T, G = oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom)
        steps = 0
        mine = batch_shard(BATCHES, rank, world)
        for k in mine:
            mu = w.spectrum_muons(1, N_BATCH, "gauss", batch=k)
            r = oracle.transport(T, G, mu.pos_q, mu.mom, wl.seed, id_base=k * N_BATCH, threads=1)
            steps += int(r["steps"].sum())
            np.savez(os.path.join(out_dir, "batch%d_rank%d.npz" % (k, rank)), pos=r["pos"], mom=r["mom"], flag=r["flag"],
                     steps=r["steps"])
        times, totals = reduce_job([1.0 + rank], [steps, N_BATCH * len(mine), len(mine)], dist)
        np.savez(os.path.join(out_dir, "job_rank%d.npz" % rank), times=times, totals=totals)
    finally:
        dist.destroy_process_group()


def test_two_rank_batch_job_equals_the_unsharded_one(tmp_path, oracle, workloads):
    world = 2
    mp.spawn(_batch_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    files = sorted(f for f in os.listdir(tmp_path) if f.startswith("batch"))
    assert files == ["batch%d_rank%d.npz" % (k, k % world) for k in range(BATCHES)]     # every batch once, on its rank
    wl = workloads.config1(n=8, n_draws=20_000)
    T, G = oracle.OracleTables(wl.hist), oracle.OracleGeometry(wl.geom)
    total_steps = 0
    for k in range(BATCHES):                           # the unsharded job: the same batches one after the other
        mu = workloads.spectrum_muons(1, N_BATCH, "gauss", batch=k)
        ref = oracle.transport(T, G, mu.pos_q, mu.mom, wl.seed, id_base=k * N_BATCH, threads=1)
        got = np.load(os.path.join(tmp_path, "batch%d_rank%d.npz" % (k, k % world)))
        for name in ("pos", "mom", "flag", "steps"):
            assert np.array_equal(got[name], ref[name]), (k, name)
        total_steps += int(ref["steps"].sum())
    for r in range(world):
        job = np.load(os.path.join(tmp_path, "job_rank%d.npz" % r))
        assert list(job["times"]) == [2.0]                                           # max over ranks
        assert list(job["totals"]) == [float(total_steps), float(N_BATCH * BATCHES), float(BATCHES)]
