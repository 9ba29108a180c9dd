"""N>1 path on CPU: world_size-2 gloo. Shards cover every pair exactly once, are balanced, and the one exchange
(all-reduce of the distance matrix) reassembles the full matrix. Per-rank distances come from the oracle here
(tests may call it); on GPUs each rank runs qp_posteriors on the same shard (bench.py --gpus N)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as td
import torch.multiprocessing as mp

from paper_1512_07437_b200 import inputs, multi


def test_shards_partition_and_balance():
    fam = inputs.config_family(4)          # log-uniform lengths: the skewed case
    pairs = inputs.all_pairs(fam.k)
    L = fam.lengths
    cells = L[pairs[:, 0]] * L[pairs[:, 1]]
    for world in (1, 2, 3, 8):
        got = np.concatenate([multi.shard_pairs(pairs, L, world, r) for r in range(world)])
        assert sorted(got.tolist()) == list(range(len(pairs)))
        loads = np.array([cells[multi.shard_pairs(pairs, L, world, r)].sum() for r in range(world)])
        assert loads.max() - loads.min() <= cells.max()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    td.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import qp_oracle as orc
    prm = inputs.default_params()
    fam = inputs.config_family(0)
    sh = multi.ShardedFamily(fam.lengths, inputs.all_pairs(fam.k), world, rank)   # the class bench.py --gpus N uses

    def run_shard(pairs):     # stands in for qp_posteriors on this rank's GPU
        run = orc.Run(prm, fam, pairs, threads=1)
        D = torch.zeros((fam.k, fam.k), dtype=torch.float64)
        D[pairs[:, 0], pairs[:, 1]] = torch.from_numpy(run.dist)
        D[pairs[:, 1], pairs[:, 0]] = torch.from_numpy(run.dist)
        return D

    full = sh.step(run_shard)
    again = sh.step(run_shard, exchange_buffer=torch.empty_like(full))             # reusable, with a caller's buffer
    assert torch.equal(full, again)
    if rank == 0:
        np.save(out, full.numpy())
    td.destroy_process_group()


def test_world2_gloo_distance_exchange(tmp_path):
    out = str(tmp_path / "D.npy")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    from oracle import qp_oracle as orc
    prm = inputs.default_params()
    fam = inputs.config_family(0)
    ref = orc.Run(prm, fam, inputs.all_pairs(fam.k)).dist_matrix()
    np.testing.assert_array_equal(np.load(out), ref)
