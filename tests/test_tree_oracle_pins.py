"""Pins of the stage-II oracle (oracle/qp_tree.py): weighted UPGMA guide tree and the tree-guided
distance. None of them re-types the oracle's own formula: a hand-worked example, scipy's
independent `weighted` linkage, ultrametric / leaf-set properties, brute force over leaf sets."""
import itertools

import numpy as np
import pytest
from scipy.cluster.hierarchy import cophenet, linkage
from scipy.spatial.distance import squareform

from oracle import qp_tree


def _rand_dyadic(rng, k):
    """symmetric integer distances: every WPGMA average of up to 2^12 of them is exact in fp32 and fp64 alike"""
    a = rng.permutation(k * (k - 1) // 2).astype(np.float64) + 1.0   # all distinct -> no ties
    return squareform(a)


def test_hand_worked_four_leaves():
    # textbook-style example worked by hand: d(a,b)=2 is the closest pair -> u=(a,b) at height 2;
    # d(u,c) = (6+8)/2 = 7, d(u,d) = (10+12)/2 = 11, d(c,d) = 9 -> merge (u,c) at 7: v; d(v,d) = (11+9)/2 = 10 -> root at 10
    D = np.array([[0, 2, 6, 10], [2, 0, 8, 12], [6, 8, 0, 9], [10, 12, 9, 0]], dtype=np.float64)
    merge, height, leaves, parent = qp_tree.wpgma(D)
    assert merge.tolist() == [[0, 1], [4, 2], [5, 3]]
    assert height.tolist() == [2.0, 7.0, 10.0]
    assert leaves.tolist() == [1, 1, 1, 1, 2, 3, 4]
    assert parent.tolist() == [4, 4, 5, 6, 5, 6, -1]
    T = qp_tree.tree_distance(leaves, parent, 4)
    # subtree node counts: (a,b) -> 3 nodes; anything with c -> 5; anything with d -> 7
    assert T.tolist() == [[1, 3, 5, 7], [3, 1, 5, 7], [5, 5, 1, 7], [7, 7, 7, 1]]


@pytest.mark.parametrize("k,seed", [(5, 0), (12, 1), (30, 2), (64, 3)])
def test_matches_scipy_weighted_linkage(k, seed):
    """scipy's linkage(method='weighted') is an independent WPGMA: same heights (as a multiset and in merge order) and
    the same cophenetic matrix (= height of the LCA of every leaf pair), which fixes the topology."""
    rng = np.random.default_rng(seed)
    D = _rand_dyadic(rng, k)
    merge, height, leaves, parent = qp_tree.wpgma(D)
    Z = linkage(squareform(D), method="weighted")
    np.testing.assert_array_equal(np.sort(height.astype(np.float64)), np.sort(Z[:, 2]))
    # cophenetic distances from the oracle's tree: height of the LCA
    coph = np.zeros((k, k))
    for x, y in itertools.combinations(range(k), 2):
        ax = set()
        a = x
        while a != -1:
            ax.add(a)
            a = int(parent[a])
        b = y
        while b not in ax:
            b = int(parent[b])
        coph[x, y] = coph[y, x] = height[b - k]
    np.testing.assert_array_equal(squareform(coph), cophenet(Z))
    np.testing.assert_array_equal(np.sort(leaves[k:]), np.sort(Z[:, 3].astype(int)))


def test_tree_distance_is_subtree_node_count_by_leaf_sets():
    """brute force: collect the leaf set under every internal node; the tree distance of x, y is 2|S|-1 for the
    smallest such set containing both."""
    rng = np.random.default_rng(7)
    k = 17
    merge, height, leaves, parent = qp_tree.wpgma(_rand_dyadic(rng, k))
    sets = {x: {x} for x in range(k)}
    for t, (a, b) in enumerate(merge):
        sets[k + t] = sets[int(a)] | sets[int(b)]
        assert len(sets[k + t]) == leaves[k + t]
    T = qp_tree.tree_distance(leaves, parent, k)
    for x in range(k):
        for y in range(k):
            want = 1 if x == y else min(2 * len(s) - 1 for s in sets.values() if x in s and y in s)
            assert T[x, y] == want
    assert (T == T.T).all() and T.max() == 2 * k - 1


def test_heights_monotone_and_ties_break_lexicographically():
    rng = np.random.default_rng(9)
    D = _rand_dyadic(rng, 20)
    _, height, _, _ = qp_tree.wpgma(D)
    assert (np.diff(height) >= 0).all()          # WPGMA is monotone (reducible linkage)
    # all distances equal: every merge is a tie; the rule picks slots (0,1), then (0,2), ... : a caterpillar
    k = 6
    merge, height, leaves, _ = qp_tree.wpgma(np.ones((k, k)) - np.eye(k))
    assert merge.tolist() == [[0, 1], [6, 2], [7, 3], [8, 4], [9, 5]] and (height == 1).all()
    assert leaves[k:].tolist() == [2, 3, 4, 5, 6]
