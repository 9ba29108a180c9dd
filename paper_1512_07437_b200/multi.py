"""Multi-GPU: the pair list shards (pairs are independent), the only exchange is the k x k distance matrix.

SURVEY.md 8(e): partition the pair list across ranks by balanced sum of n*m, replicate the (small) sequences and
parameters, run qp_posteriors per rank on its shard, then one all-reduce-sum of the zero-initialised distance
matrix over NCCL (every entry is written by exactly one rank). CSR output stays sharded by pair. There is no
collective inside the DP, so there is nothing to fuse a kernel with.
"""
from __future__ import annotations

import numpy as np


def shard_assignment(cells: np.ndarray, world: int) -> np.ndarray:
    """rank of every pair: sort by cells (largest first, stable), deal in boustrophedon order
    0,1,..,W-1,W-1,..,1,0,... Deterministic; the per-rank cell sums differ by at most ~one large pair."""
    order = np.argsort(-np.asarray(cells, dtype=np.int64), kind="stable")
    j = np.arange(len(order)) % (2 * world)
    r = np.where(j < world, j, 2 * world - 1 - j)
    rank = np.empty(len(order), dtype=np.int32)
    rank[order] = r
    return rank


def shard_pairs(pairs: np.ndarray, lengths: np.ndarray, world: int, rank: int) -> np.ndarray:
    """Indices (into `pairs`, ascending) of the pairs owned by `rank`."""
    pairs = np.asarray(pairs).reshape(-1, 2)
    cells = lengths[pairs[:, 0]].astype(np.int64) * lengths[pairs[:, 1]].astype(np.int64)
    return np.nonzero(shard_assignment(cells, world) == rank)[0]


def exchange_distances(dist, group=None):
    """The one exchange step: sum the per-rank k x k matrices (disjoint supports) in place. torch tensor, any backend."""
    import torch.distributed as td
    if td.is_available() and td.is_initialized() and td.get_world_size(group) > 1:
        td.all_reduce(dist, op=td.ReduceOp.SUM, group=group)
    return dist


class ShardedFamily:
    """One family over `world` ranks: this rank's slice of the pair list, and one step of the path =
    run the posterior stage on the slice (a callback: qp_posteriors on a GPU, anything that fills this rank's entries
    of the k x k matrix elsewhere) followed by the one exchange. bench.py and tests/test_multi_gloo.py both go
    through this class."""

    def __init__(self, lengths, all_pairs, world, rank):
        self.world, self.rank = int(world), int(rank)
        self.all_pairs = np.ascontiguousarray(all_pairs, dtype=np.int32).reshape(-1, 2)
        self.mine = shard_pairs(self.all_pairs, np.asarray(lengths), self.world, self.rank)
        self.pairs = np.ascontiguousarray(self.all_pairs[self.mine])

    def step(self, run_shard, exchange_buffer=None, group=None):
        """run_shard(pairs) -> k x k torch tensor holding this rank's distances (zeros elsewhere). Returns the full
        matrix (summed over ranks). `exchange_buffer`: optional tensor of the same shape to reduce in (the result of
        run_shard is left untouched, e.g. because the next step rewrites it in place)."""
        d = run_shard(self.pairs)
        buf = d.clone() if exchange_buffer is None else exchange_buffer.copy_(d)
        return exchange_distances(buf, group)
