"""GPU parity of stage II (qp_guide_tree through the C ABI) against oracle/qp_tree.py: bit-exact merges, heights,
leaf counts, parents and tree distances (integer / index work; the fp32 averages are the same IEEE operations on both
sides)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import qp_oracle as orc
from oracle import qp_tree
from paper_1512_07437_b200 import inputs


def _run(D):
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1512_07437_b200 import qp
    t = qp.guide_tree(torch.from_numpy(np.ascontiguousarray(D, dtype=np.float32)).cuda())
    torch.cuda.synchronize()
    return t


def _check(D):
    k = D.shape[0]
    t = _run(D)
    merge, height, leaves, parent = qp_tree.wpgma(D)
    assert np.array_equal(t.merge.cpu().numpy(), merge)
    assert np.array_equal(t.height.cpu().numpy(), height)
    assert np.array_equal(t.leaves.cpu().numpy(), leaves)
    assert np.array_equal(t.parent.cpu().numpy(), parent)
    if k <= 400:
        assert np.array_equal(t.treedist.cpu().numpy(), qp_tree.tree_distance(leaves, parent, k))
    else:   # the oracle's pairwise walk is slow: sampled pairs + properties that hold for every pair
        T = t.treedist.cpu().numpy()
        rng = np.random.default_rng(0)
        idx = rng.integers(0, k, size=(300, 2))
        anc = lambda x: [a for a in iter(lambda s=[x]: s.append(int(parent[s[-1]])) or s[-2] if s[-1] != -1 else None, None)]
        for x, y in idx:
            ax = set(anc(int(x)))
            b = int(y)
            while b not in ax:
                b = int(parent[b])
            assert T[x, y] == (2 * leaves[b] - 1 if x != y else 1)
        assert (T == T.T).all() and (np.diag(T) == 1).all() and T.max() == 2 * k - 1 and (T % 2 == 1).all()


@pytest.mark.parametrize("k,seed", [(1, 0), (2, 0), (3, 1), (8, 2), (33, 3), (200, 4)])
def test_random_matrices(k, seed):
    rng = np.random.default_rng(seed)
    A = rng.random((k, k)).astype(np.float32)
    D = np.triu(A, 1) + np.triu(A, 1).T
    _check(D)


def test_ties_everywhere():
    """few distinct values: nearly every step is a tie, the lexicographic rule decides"""
    rng = np.random.default_rng(5)
    k = 70
    A = rng.integers(1, 4, size=(k, k)).astype(np.float32) * 0.25
    _check(np.triu(A, 1) + np.triu(A, 1).T)
    _check(np.ones((40, 40), dtype=np.float32) - np.eye(40, dtype=np.float32))


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_guide_tree_of_the_posterior_stage(default_params, cfg):
    """the distance matrix that qp_posteriors writes for configs[cfg] -> guide tree, against the oracle on the SAME
    matrix (configs[3]: k = 1000)"""
    import torch
    from paper_1512_07437_b200 import qp
    fam = inputs.config_family(cfg)
    pairs = inputs.all_pairs(fam.k)
    res = qp.run_family(fam, pairs, default_params)
    D = res.dist.cpu().numpy()
    del res
    torch.cuda.empty_cache()
    _check(D)
