"""Pins for oracle/qp_oracle.c against things other than itself (pins 1-12).

CPU only. Each test names the pin and what a plausible mistake would break.
"""
import math

import numpy as np
import pytest

from oracle import qp_oracle as orc
from paper_1512_07437_b200 import inputs
from tests import bruteforce as bf

LOG = math.log


def _rand_seq(rng, n, A):
    return rng.integers(0, A, size=n).astype(np.uint8)


# ---- pin 1: brute-force path enumeration --------------------------------------------------------------------
@pytest.mark.parametrize("G", [1, 2])
@pytest.mark.parametrize("shape", [(1, 1), (1, 2), (2, 1), (1, 4), (3, 1), (2, 3), (3, 3), (4, 5), (5, 4), (5, 5)])
def test_pin1_bruteforce_posterior_and_logZ(G, shape):
    n, m = shape
    rng = np.random.default_rng(1000 * G + 10 * n + m)
    for trial in range(3):
        model = inputs.random_model(rng, G, alphabet=4)
        x, y = _rand_seq(rng, n, 4), _rand_seq(rng, m, 4)
        P_bf, Z_bf = bf.posterior(model, x, y)
        P, zf, zb, F, B = orc.posterior(model, x, y)
        assert zf == pytest.approx(LOG(Z_bf), rel=1e-12, abs=1e-12)
        assert zb == pytest.approx(LOG(Z_bf), rel=1e-12, abs=1e-12)
        np.testing.assert_allclose(P, np.array(P_bf), rtol=1e-11, atol=1e-14)


def test_pin1_bruteforce_6x6_default_like_models():
    rng = np.random.default_rng(66)
    x, y = _rand_seq(rng, 6, 20), _rand_seq(rng, 6, 20)
    for model in (inputs.default_pf(), inputs.default_hmm()):
        P_bf, Z_bf = bf.posterior(model, x, y)
        P, zf, zb, _, _ = orc.posterior(model, x, y)
        assert zf == pytest.approx(LOG(Z_bf), rel=1e-12)
        np.testing.assert_allclose(P, np.array(P_bf), rtol=1e-10, atol=1e-15)


def test_pin1_bruteforce_mea_and_distance():
    rng = np.random.default_rng(7)
    for n, m in [(1, 1), (2, 5), (4, 4), (5, 3), (6, 6)]:
        P = rng.random((n, m)) ** 3
        a = orc.mea(P)
        assert a == pytest.approx(bf.mea(P.tolist()), rel=1e-13)
        assert orc.distance(a, n, m) == pytest.approx(1.0 - a / min(n, m), rel=1e-15)


def test_mea_known_values():
    # hand-checkable: identity matrix -> n ; anti-diagonal ones -> 1 ; a single row takes its max
    assert orc.mea(np.eye(5)) == 5.0
    assert orc.mea(np.fliplr(np.eye(5))) == 1.0
    assert orc.mea(np.array([[0.1, 0.7, 0.3]])) == 0.7
    # crossing matches cannot both be used: best is 0.9, not 0.8+0.9
    assert orc.mea(np.array([[0.0, 0.8], [0.9, 0.0]])) == pytest.approx(0.9)
    assert orc.mea(np.array([[0.5, 0.0], [0.0, 0.6]])) == pytest.approx(1.1)


def test_combine_rms_known_values():
    out = orc.combine(np.array([0.6, 0.3, 0.0, 1.0]), np.array([0.8, 0.3, 0.5, 1.0]))
    np.testing.assert_allclose(out, [math.sqrt(0.5), 0.3, 0.5 / math.sqrt(2), 1.0], rtol=1e-15)


# ---- pin 2 / 3: totals and the row/column marginal identity over ALL state planes -----------------------------
@pytest.mark.parametrize("which", ["hmm", "pf", "rand1", "rand2"])
def test_pin2_pin3_totals_and_marginals(which):
    rng = np.random.default_rng(23)
    model = {"hmm": inputs.default_hmm(), "pf": inputs.default_pf(),
             "rand1": inputs.random_model(rng, 1, 20), "rand2": inputs.random_model(rng, 2, 20)}[which]
    x, y = _rand_seq(rng, 37, 20), _rand_seq(rng, 52, 20)
    P, zf, zb, F, B = orc.posterior(model, x, y)
    assert zb == pytest.approx(zf, rel=1e-12)
    G = model.n_ins
    n, m = len(x), len(y)
    with np.errstate(over="ignore"):
        post = np.exp(F + B - zf)  # all planes, (n+1) x (m+1)
    # each path consumes x_i exactly once: in M at (i, j>=1) or in some X_g at (i, j>=0)
    rows = post[0, 1:, 1:].sum(axis=1) + sum(post[1 + g, 1:, :].sum(axis=1) for g in range(G))
    cols = post[0, 1:, 1:].sum(axis=0) + sum(post[1 + G + g, :, 1:].sum(axis=0) for g in range(G))
    np.testing.assert_allclose(rows, np.ones(n), rtol=1e-10)
    np.testing.assert_allclose(cols, np.ones(m), rtol=1e-10)
    assert (P.sum(axis=1) <= 1 + 1e-9).all() and (P.sum(axis=0) <= 1 + 1e-9).all() and (P >= 0).all()


# ---- pin 4: transposition ----------------------------------------------------------------------------------
def test_pin4_transposition(default_params):
    rng = np.random.default_rng(4)
    x, y = _rand_seq(rng, 31, 20), _rand_seq(rng, 44, 20)
    a, b = orc.pair(default_params, x, y), orc.pair(default_params, y, x)
    np.testing.assert_allclose(a.P, b.P.T, rtol=1e-11, atol=1e-300)
    np.testing.assert_allclose(a.Ph, b.Ph.T, rtol=1e-11, atol=1e-300)
    assert a.dist == pytest.approx(b.dist, abs=1e-13)
    np.testing.assert_allclose(a.logZ, b.logZ, rtol=1e-12)


# ---- pin 5 / 6: closed forms ----------------------------------------------------------------------------------
def test_pin5_one_by_one(default_params):
    r = orc.pair(default_params, np.array([3], np.uint8), np.array([11], np.uint8))
    assert r.P[0, 0] == pytest.approx(1.0, abs=1e-14) and r.dist == pytest.approx(0.0, abs=1e-14)
    assert r.Ph[0, 0] == pytest.approx(1.0, abs=1e-14) and r.Pp[0, 0] == pytest.approx(1.0, abs=1e-14)


def test_pin6_one_by_two_closed_forms():
    pf, hmm = inputs.default_pf(), inputs.default_hmm()
    q = inputs.background()
    for (x1, y1, y2) in [(0, 0, 5), (7, 3, 7), (19, 19, 19), (2, 9, 4)]:
        x, y = np.array([x1], np.uint8), np.array([y1, y2], np.uint8)
        # PF: the two alignments differ only in which y pairs with x1: logistic in (s(x1,y2)-s(x1,y1))/T
        P, _, _, _, _ = orc.posterior(pf, x, y)
        d = pf.log_match[x1, y2] - pf.log_match[x1, y1]  # already divided by T
        assert P[0, 0] == pytest.approx(1.0 / (1.0 + math.exp(d)), rel=1e-12)
        assert P[0, 1] == pytest.approx(1.0 - P[0, 0], rel=1e-12)
        # HMM: paths M Y_g (x1~y1) and Y_g M (x1~y2)
        e = np.exp(hmm.log_match)
        piM, pi = math.exp(hmm.init_M), np.exp(hmm.init_I)
        dl, ep = np.exp(hmm.t_MI), np.exp(hmm.t_II)
        a = sum(piM * e[x1, y1] * dl[g] * q[y2] * pi[g] for g in range(2))           # end weight = init weight
        b = sum(pi[g] * q[y1] * (1 - ep[g]) * e[x1, y2] * piM for g in range(2))
        Ph, _, _, _, _ = orc.posterior(hmm, x, y)
        assert Ph[0, 0] == pytest.approx(a / (a + b), rel=1e-12)
        assert Ph[0, 1] == pytest.approx(b / (a + b), rel=1e-12)


# ---- pin 7: nnz bound, CSR vs dense --------------------------------------------------------------------------
def test_pin7_nnz_bound_and_csr_consistency(default_params):
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)[:6]
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    tau = default_params.threshold
    for p in range(len(pairs)):
        P = run.dense(p)
        rp, col, val = run.csr(p)
        n, m = P.shape
        assert len(rp) == n + 1 and rp[0] == 0 and rp[-1] == len(col) == run.nnz[p]
        assert (np.diff(rp) <= min(m, math.floor(2.0 / tau))).all()
        ii, jj = np.nonzero(P >= tau)
        np.testing.assert_array_equal(col, jj)
        np.testing.assert_array_equal(np.repeat(np.arange(n), np.diff(rp)), ii)
        np.testing.assert_array_equal(val, P[ii, jj])  # values unmodified
        single = orc.pair(default_params, fam.seq(pairs[p, 0]), fam.seq(pairs[p, 1]))
        assert run.dist[p] == single.dist
        np.testing.assert_array_equal(run.logZ(p), single.logZ)
    D = run.dist_matrix()
    assert (D == D.T).all() and (D >= 0).all() and (D <= 1).all()


# ---- pin 8: background normalisation leaves P unchanged --------------------------------------------------------
def test_pin8_background_normalisation_invariance():
    hmm = inputs.default_hmm()
    rng = np.random.default_rng(8)
    x, y = _rand_seq(rng, 40, 20), _rand_seq(rng, 33, 20)
    P0, z0, _, _, _ = orc.posterior(hmm, x, y)
    lx = hmm.log_ins
    norm = inputs.Model(**{**hmm.__dict__, "log_match": hmm.log_match - lx[:, None] - lx[None, :],
                           "log_ins": np.zeros_like(lx)})
    P1, z1, _, _, _ = orc.posterior(norm, x, y)
    np.testing.assert_allclose(P1, P0, rtol=1e-10, atol=1e-300)
    assert z0 == pytest.approx(z1 + lx[x].sum() + lx[y].sum(), rel=1e-12)


# ---- pin 9: PF reversal symmetry ---------------------------------------------------------------------------------
def test_pin9_pf_reversal_symmetry():
    pf = inputs.default_pf()
    rng = np.random.default_rng(9)
    x, y = _rand_seq(rng, 29, 20), _rand_seq(rng, 35, 20)
    P, z, _, _, _ = orc.posterior(pf, x, y)
    Pr, zr, _, _, _ = orc.posterior(pf, x[::-1].copy(), y[::-1].copy())
    np.testing.assert_allclose(Pr[::-1, ::-1], P, rtol=1e-10, atol=1e-300)
    assert z == pytest.approx(zr, rel=1e-12)


# ---- pin 10: T -> 0 limit is the unique optimal Gotoh alignment ----------------------------------------------------
def _gotoh(S, go, ge, x, y):
    """Textbook global affine-gap alignment (gap of length L costs go+(L-1)ge, terminal gaps charged).
    Returns (score, set of matched (i,j) 1-based)."""
    n, m = len(x), len(y)
    NEG = -1e300
    M = np.full((n + 1, m + 1), NEG); X = M.copy(); Y = M.copy()
    M[0, 0] = 0.0
    for i in range(1, n + 1):
        X[i, 0] = -go - (i - 1) * ge
    for j in range(1, m + 1):
        Y[0, j] = -go - (j - 1) * ge
    for i in range(1, n + 1):
        for j in range(1, m + 1):
            M[i, j] = S[x[i - 1], y[j - 1]] + max(M[i - 1, j - 1], X[i - 1, j - 1], Y[i - 1, j - 1])
            X[i, j] = max(M[i - 1, j] - go, X[i - 1, j] - ge)      # no Y->X
            Y[i, j] = max(M[i, j - 1] - go, Y[i, j - 1] - ge)      # no X->Y
    st = int(np.argmax([M[n, m], X[n, m], Y[n, m]]))
    score = [M[n, m], X[n, m], Y[n, m]][st]
    i, j, cells = n, m, set()
    while i > 0 or j > 0:
        if st == 0:
            cells.add((i, j))
            st = int(np.argmax([M[i - 1, j - 1], X[i - 1, j - 1], Y[i - 1, j - 1]]))
            i, j = i - 1, j - 1
        elif st == 1:
            st = 0 if (i == 1 and j == 0) or (i > 1 and M[i - 1, j] - go >= X[i - 1, j] - ge) else 1
            i -= 1
        else:
            st = 0 if (j == 1 and i == 0) or (j > 1 and M[i, j - 1] - go >= Y[i, j - 1] - ge) else 2
            j -= 1
    return score, cells


def test_pin10_zero_temperature_limit_is_gotoh():
    rng = np.random.default_rng(10)
    A = 20
    S = rng.normal(0, 2.0, size=(A, A)); S = 0.5 * (S + S.T) + 2.0 * np.eye(A)
    go, ge, T = 2.3, 0.7, 0.002
    for n, m in [(9, 12), (14, 10), (12, 12)]:
        # residues distinct within each sequence: no two alignments can tie exactly, so the optimum is unique
        x, y = rng.permutation(A)[:n].astype(np.uint8), rng.permutation(A)[:m].astype(np.uint8)
        score, cells = _gotoh(S, go, ge, x, y)
        pf = inputs.Model(n_ins=1, alphabet=A, log_match=S / T, log_ins=np.zeros(A), t_MM=0.0,
                          t_MI=(-go / T,), t_II=(-ge / T,), t_IM=(0.0,), init_M=0.0, init_I=(-go / T,),
                          end_M=0.0, end_I=(0.0,))
        P, zf, _, _, _ = orc.posterior(pf, x, y)
        ind = np.zeros((n, m))
        for (i, j) in cells:
            ind[i - 1, j - 1] = 1.0
        np.testing.assert_allclose(P, ind, atol=1e-3)       # unique optimum (continuous random scores)
        assert zf * T == pytest.approx(score, abs=5 * T)     # T log Z -> optimal score


# ---- pin 11 / 12: identical sequences, ranges -----------------------------------------------------------------------
def test_pin11_identical_sequences(default_params):
    rng = np.random.default_rng(11)
    x = rng.choice(20, size=50, p=inputs.background()).astype(np.uint8)
    r = orc.pair(default_params, x, x)
    assert (np.diag(r.P)[5:-5] > 0.9).all() and r.dist < 0.1


def test_pin12_ranges_on_cfg0(default_params):
    fam = inputs.config_family(0)
    for (a, b) in [(0, 1), (2, 7), (3, 4)]:
        r = orc.pair(default_params, fam.seq(a), fam.seq(b))
        n, m = r.P.shape
        A = (1.0 - r.dist) * min(n, m)
        assert 0.0 <= r.dist <= 1.0 and A <= min(n, m) + 1e-9 and A >= r.P.max() - 1e-12
        # c-4 #14: per-model rows in [0,1]; RMS-combined rows bounded by sqrt(2)
        assert r.Ph.sum(1).max() <= 1 + 1e-9 and r.Pp.sum(1).max() <= 1 + 1e-9
        assert r.P.sum(1).max() <= math.sqrt(2) + 1e-9
        assert r.logZ[0] == pytest.approx(r.logZ[1], rel=1e-12) and r.logZ[2] == pytest.approx(r.logZ[3], rel=1e-12)
