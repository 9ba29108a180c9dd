"""Pins of the stage-III oracle (oracle/qp_consistency.py) against things other than itself: the textbook consistency
transformation written as ONE block-matrix product, exact fixed points, hand-computed numbers, hand-listed selections.
A plausible slip -- a dropped z, the wrong normaliser, a transposed operand, a missing factor 2, a wrong end point of
h_xy -- fails at least one of them. CPU only."""
import numpy as np
import pytest
import scipy.sparse as sp

from oracle import qp_consistency as oc


def _all_pairs(k):
    return [(x, y) for x in range(k) for y in range(x + 1, k)]


def _dense_family(rng, lens):
    """Random strictly positive dense matrices for every pair x < y (so that masking and thresholding are inert)."""
    return {(x, y): sp.csr_matrix(rng.uniform(0.05, 1.0, size=(lens[x], lens[y]))) for (x, y) in _all_pairs(len(lens))}


def _far(k):
    return np.full((k, k), 10 ** 6, dtype=np.int64)


def test_full_consistency_equals_block_matrix_square():
    """PAPER.md:53 relaxation, R1 with h = 1 and every z selected == the textbook transformation
    S'_xy = (1/k) sum_z S_xz S_zy over ALL k sequences with S_xx = I, S_zx = S_xz^T: assemble the N x N block matrix B
    (N = total residues) and read S' off B @ B / k. One numpy product, no per-pair loop, no selection code."""
    rng = np.random.default_rng(1)
    lens = [3, 5, 2, 4, 6]
    k = len(lens)
    S = _dense_family(rng, lens)
    off = np.concatenate([[0], np.cumsum(lens)])
    B = np.zeros((off[-1], off[-1]))
    for x in range(k):
        B[off[x]:off[x + 1], off[x]:off[x + 1]] = np.eye(lens[x])
    for (x, y), M in S.items():
        B[off[x]:off[x + 1], off[y]:off[y + 1]] = M.toarray()
        B[off[y]:off[y + 1], off[x]:off[x + 1]] = M.toarray().T
    BB = B @ B / k
    out, cnt = oc.transform(S, k, np.ones((k, k), dtype=np.int64), T=1, h=1.0, tau=0.0)
    for (x, y) in S:
        assert cnt[(x, y)] == k - 2
        np.testing.assert_allclose(out[(x, y)].toarray(), BB[off[x]:off[x + 1], off[y]:off[y + 1]], rtol=1e-13, atol=1e-15)


@pytest.mark.parametrize("h", [1.0, 3.0])
def test_transitive_alignments_are_a_fixed_point(h):
    """S_xy = Pi_x^T Pi_y for permutation matrices Pi: S_xz S_zy = S_xy for every z, so R1 gives S' = S exactly for any
    h and any selection. The matrices are not symmetric, so a transposed operand, a dropped term or a wrong
    normaliser all break the identity."""
    rng = np.random.default_rng(2)
    k, n = 6, 7
    Pi = [np.eye(n)[rng.permutation(n)] for _ in range(k)]
    S = {(x, y): sp.csr_matrix(Pi[x].T @ Pi[y]) for (x, y) in _all_pairs(k)}
    td = rng.integers(1, 12, size=(k, k))
    td = np.maximum(td, td.T)
    for T in (0, 6, 100):
        out, cnt = oc.transform(S, k, td, T=T, h=h, tau=0.01)
        for key in S:
            np.testing.assert_allclose(out[key].toarray(), S[key].toarray(), rtol=0, atol=1e-15)
    assert any(c > 0 for c in cnt.values())


def test_no_selected_sequence_leaves_the_matrix_alone():
    rng = np.random.default_rng(3)
    S = _dense_family(rng, [4, 3, 5, 2])
    out, cnt = oc.transform(S, 4, _far(4), T=200, h=3.0, tau=0.0)
    assert all(c == 0 for c in cnt.values())
    for key in S:
        assert np.array_equal(out[key].toarray(), S[key].toarray())


def test_hand_computed_scalars():
    """Three sequences of one residue: S_01 = 0.5, S_02 = 0.4, S_12 = 0.8, every z selected, h = 3, R = 200:
    h_01 = 1 + 2/200 = 1.01; S'_01 = (2*1.01*0.5 + 0.4*0.8) / (2*1.01 + 1) = 1.33 / 3.02;
    S'_02 = (2*1.01*0.4 + 0.5*0.8) / 3.02 = 1.208 / 3.02;  S'_12 = (2*1.01*0.8 + 0.5*0.4) / 3.02 = 1.816 / 3.02."""
    S = {(0, 1): sp.csr_matrix([[0.5]]), (0, 2): sp.csr_matrix([[0.4]]), (1, 2): sp.csr_matrix([[0.8]])}
    out, cnt = oc.transform(S, 3, np.ones((3, 3), dtype=np.int64), T=200, h=3.0, max_relax=200, tau=0.01)
    assert cnt == {(0, 1): 1, (0, 2): 1, (1, 2): 1}
    assert out[(0, 1)][0, 0] == pytest.approx(1.33 / 3.02, rel=1e-15)
    assert out[(0, 2)][0, 0] == pytest.approx(1.208 / 3.02, rel=1e-15)
    assert out[(1, 2)][0, 0] == pytest.approx(1.816 / 3.02, rel=1e-15)


def test_h_coefficient_end_points():
    """1 with no relaxation, h at the maximum number of relaxations (200); R2: linear in between."""
    assert oc.h_coefficient(0, 3.0, 200) == 1.0
    assert oc.h_coefficient(200, 3.0, 200) == 3.0
    assert oc.h_coefficient(1000, 3.0, 200) == 3.0
    assert oc.h_coefficient(100, 3.0, 200) == 2.0
    assert oc.h_coefficient(50, 1.0, 200) == 1.0


def test_selection_on_a_hand_made_tree():
    """PAPER.md:63 Figure 2 in small: leaves x=0, y=1, z=2 under one node of size 5 (x, y under a node of size 3),
    u=3 joins at the root (size 7). Tree-guided distances (node counts): d01 = 3, d02 = d12 = 5, d*3 = 7.
    T = 5 with f = max accepts z and rejects u; f = sum needs T >= 10 for z; f = min accepts z for (0,1) at T = 5."""
    td = np.array([[1, 3, 5, 7], [3, 1, 5, 7], [5, 5, 1, 7], [7, 7, 7, 1]])
    S = {p: sp.csr_matrix(np.ones((1, 1))) for p in _all_pairs(4)}
    assert oc.select(S, 4, td, 0, 1, T=5, f=oc.SEL_MAX) == [2]
    assert oc.select(S, 4, td, 0, 1, T=4, f=oc.SEL_MAX) == []
    assert oc.select(S, 4, td, 0, 1, T=7, f=oc.SEL_MAX) == [2, 3]
    assert oc.select(S, 4, td, 0, 2, T=5, f=oc.SEL_MAX) == [1]          # d01 = 3, d21 = 5
    assert oc.select(S, 4, td, 0, 1, T=9, f=oc.SEL_SUM) == []
    assert oc.select(S, 4, td, 0, 1, T=10, f=oc.SEL_SUM) == [2]
    assert oc.select(S, 4, td, 0, 2, T=3, f=oc.SEL_MIN) == [1]          # min(d01, d21) = 3
    assert oc.select(S, 4, td, 0, 3, T=6, f=oc.SEL_MIN) == [1, 2]       # min(d01, d31) = 3, min(d02, d32) = 5
    del S[(1, 2)]                                                        # R3: a missing pair is never relaxed over
    assert oc.select(S, 4, td, 0, 1, T=7, f=oc.SEL_MAX) == [3]


def test_listing_a_pair_the_other_way_round_gives_the_transpose():
    rng = np.random.default_rng(4)
    lens = [3, 4, 5, 2]
    S = _dense_family(rng, lens)
    td = np.ones((4, 4), dtype=np.int64)
    out, _ = oc.transform(S, 4, td, T=5, h=3.0, tau=0.0)
    flipped = dict(S)
    flipped[(2, 1)] = flipped.pop((1, 2)).T.tocsr()
    out2, _ = oc.transform(flipped, 4, td, T=5, h=3.0, tau=0.0)
    np.testing.assert_allclose(out2[(2, 1)].toarray(), out[(1, 2)].toarray().T, rtol=1e-14)
    np.testing.assert_allclose(out2[(0, 3)].toarray(), out[(0, 3)].toarray(), rtol=1e-14)


def test_relabelling_the_sequences_changes_nothing():
    rng = np.random.default_rng(5)
    lens = [3, 4, 2, 5, 3]
    k = len(lens)
    S = _dense_family(rng, lens)
    td = rng.integers(1, 9, size=(k, k))
    td = np.maximum(td, td.T)
    out, cnt = oc.transform(S, k, td, T=5, h=3.0, tau=0.0)
    perm = [3, 0, 4, 1, 2]                      # new label of old sequence s
    S2 = {}
    for (x, y), M in S.items():
        a, b = perm[x], perm[y]
        S2[(a, b) if a < b else (b, a)] = M if a < b else M.T.tocsr()
    inv = np.argsort(perm)
    td2 = td[np.ix_(inv, inv)]
    out2, cnt2 = oc.transform(S2, k, td2, T=5, h=3.0, tau=0.0)
    for (x, y) in S:
        a, b = perm[x], perm[y]
        got = out2[(a, b)].toarray() if a < b else out2[(b, a)].toarray().T
        np.testing.assert_allclose(got, out[(x, y)].toarray(), rtol=1e-13)
        assert cnt2[(a, b) if a < b else (b, a)] == cnt[(x, y)]


def test_pattern_is_kept_and_small_values_are_dropped():
    """R4 by hand. S_01 = [[0.5, 0], [0, 0.02]] (two stored cells), S_02 = [[0.9], [0.9]], S_12 = [[0.9], [0.9]]:
    S_02 S_21 = 0.81 in all four cells. r = 1, h = 1: cell (0,0) -> (1.0 + 0.81)/3; cell (1,1) -> (0.04 + 0.81)/3;
    cells (0,1), (1,0) are not in S_01's pattern and must not appear. With S_02 = [[0.9], [0.0]] instead, cell (1,1)
    -> 0.04/3 = 0.0133 >= tau = 0.01 stays; with tau = 0.02 it is dropped."""
    S01 = sp.csr_matrix(np.array([[0.5, 0.0], [0.0, 0.02]]))
    td = np.ones((3, 3), dtype=np.int64)
    S = {(0, 1): S01, (0, 2): sp.csr_matrix([[0.9], [0.9]]), (1, 2): sp.csr_matrix([[0.9], [0.9]])}
    out, _ = oc.transform(S, 3, td, T=5, h=1.0, tau=0.01)
    np.testing.assert_allclose(out[(0, 1)].toarray(), [[1.81 / 3, 0.0], [0.0, 0.85 / 3]], rtol=1e-15)
    assert out[(0, 1)].nnz == 2
    S[(0, 2)] = sp.csr_matrix(np.array([[0.9], [0.0]]))
    out, _ = oc.transform(S, 3, td, T=5, h=1.0, tau=0.01)
    assert out[(0, 1)].nnz == 2 and out[(0, 1)][1, 1] == pytest.approx(0.04 / 3, rel=1e-15)
    out, _ = oc.transform(S, 3, td, T=5, h=1.0, tau=0.02)
    assert out[(0, 1)].nnz == 1 and out[(0, 1)][0, 0] == pytest.approx(1.81 / 3, rel=1e-15)


def test_number_of_transformations():
    """2 for k < 50, 1 otherwise."""
    assert oc.n_transformations(8) == 2 and oc.n_transformations(49) == 2
    assert oc.n_transformations(50) == 1 and oc.n_transformations(1000) == 1


def test_chain_from_stage_one_stays_a_probability(default_params):
    """configs[0] through the oracle chain stage I -> II -> III: relaxed values stay in [tau, 1], the pattern only
    shrinks, and the number of relaxations follows the tree distances."""
    from oracle import qp_oracle as orc
    from oracle import qp_tree
    from paper_1512_07437_b200 import inputs
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(default_params, fam, pairs)
    L = fam.lengths
    S = {(int(a), int(b)): oc.from_csr(*run.csr(p), L[a], L[b]) for p, (a, b) in enumerate(pairs)}
    merge, height, leaves, parent = qp_tree.wpgma(run.dist_matrix())
    td = qp_tree.tree_distance(leaves, parent, fam.k)
    out, cnt = oc.transform(S, fam.k, td, T=9, h=3.0, tau=default_params.threshold)
    assert 0 < sum(cnt.values()) < fam.k * (fam.k - 1) * (fam.k - 2) // 2
    for key, M in out.items():
        assert M.nnz <= S[key].nnz
        assert M.nnz == 0 or (M.data.min() >= default_params.threshold and M.data.max() <= 1.0 + 1e-12)
        assert (S[key].toarray()[M.toarray() > 0] > 0).all()
