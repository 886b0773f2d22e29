"""Multi-GPU sharding of the transport path: contiguous muon-id ranges per rank, replicated
tables and grids, no collective on the data path.  Only the bookkeeping lives here — which ids a rank owns and
how per-rank timings and totals combine into the whole-job figures bench.py prints — so that it can be tested
on CPU with the gloo backend.  PAPER.md L57 (independent histories), L184 (batches across devices).
"""
from dataclasses import dataclass


@dataclass(frozen=True)
class Shard:
    rank: int
    world: int
    id_base: int       # first global muon id of this rank
    n: int             # muons of this rank


def weak_shard(muons_per_gpu: int, rank: int, world: int) -> Shard:
    """Weak scaling (bench.py): every rank transports its own batch of `muons_per_gpu` muons."""
    if not (0 <= rank < world) or muons_per_gpu < 0:
        raise ValueError("bad shard request")
    return Shard(rank, world, rank * muons_per_gpu, muons_per_gpu)


def strong_shard(n_total: int, rank: int, world: int) -> Shard:
    """Strong scaling: `n_total` muons split into contiguous, near-equal id ranges (the first n_total % world
    ranks take one more)."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard request")
    q, r = divmod(n_total, world)
    n = q + (1 if rank < r else 0)
    return Shard(rank, world, rank * q + min(rank, r), n)


def batch_shard(n_batches: int, rank: int, world: int):
    """A job made of whole batches (BASELINE.json configs[4]: 10^8 muons as ten batches of 10^7, batch k holding the ids
    k * batch_size ..): batch k goes to rank k % world, so the ranks' batch counts differ by at most one and every batch
    is run exactly once.  Returns this rank's batch indices, ascending; its id_base for batch k is k * batch_size."""
    if not (0 <= rank < world) or n_batches < 0:
        raise ValueError("bad shard request")
    return list(range(rank, n_batches, world))


def reduce_job(times_s, totals, dist=None, device=None):
    """Whole-job figures from per-rank ones: element-wise MAX of `times_s` (device-timed seconds) and SUM of
    `totals` (muon-steps, muons, ...) over the ranks of the default process group.  Returns two lists."""
    import torch
    t = torch.tensor(list(times_s), dtype=torch.float64, device=device)
    s = torch.tensor(list(totals), dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return t.tolist(), s.tolist()


def gather_ranges(shard, dist=None, device=None):
    """[[first id, one past the last id]] of every rank, in rank order, as the ranks themselves report them."""
    import torch
    mine = torch.tensor([shard.id_base, shard.id_base + shard.n], dtype=torch.int64, device=device)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [mine.tolist()]
    parts = [torch.zeros_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, mine)
    return [p.tolist() for p in parts]
