"""GPU parity of stage III (qp_consistency, through the C ABI) against oracle/qp_consistency.py, element by element.

Both sides get THE SAME inputs, made by the oracle chain only: the stage-I CSR of oracle/qp_oracle.c with its values
rounded to fp32 (the precision stage III receives them in), and the tree-guided distances of oracle/qp_tree.py. No
input of the oracle comes from the CUDA path.

Tolerance: the kernel accumulates in fp32, one rounding per multiply-add; a cell sums at most
|sel| * min(row length) products whose total is <= |sel| (rows of S sum to <= sqrt 2), so the rounding error of the
sum is <= |sel| * sqrt(terms) * 2^-24 and, after the division by 2h + |sel|, below ~25 * 6e-8 = 1.5e-6 in the worst
case: |dS'| <= 2e-6 absolute (measured <= 4.5e-7); the relaxed pattern must equal the oracle's except where the
oracle's relaxed value lies within 2e-6 of the threshold.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import qp_consistency as oc
from oracle import qp_oracle as orc
from oracle import qp_tree
from paper_1512_07437_b200 import inputs

S_ATOL = 2e-6
BAND = 2e-6


def _qp():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1512_07437_b200 import qp
    return qp


class _Csr:
    pass


def _oracle_stage1(fam, pairs, prm):
    """Stage I + II by the oracle: {(x, y): csr with fp32-rounded values}, tree distances."""
    run = orc.Run(prm, fam, pairs)
    L = fam.lengths
    S = {}
    for p, (a, b) in enumerate(pairs):
        rp, col, val = run.csr(p)
        S[(int(a), int(b))] = oc.from_csr(rp, col, val.astype(np.float32).astype(np.float64), L[a], L[b])
    k = fam.k
    D = np.zeros((k, k))
    D[pairs[:, 0], pairs[:, 1]] = run.dist
    D[pairs[:, 1], pairs[:, 0]] = run.dist
    merge, height, leaves, parent = qp_tree.wpgma(D)
    return S, qp_tree.tree_distance(leaves, parent, k)


def _upload(S, pairs, fam, dev):
    import torch
    L = fam.lengths
    rb, nb, rps, cols, vals = [0], [0], [], [], []
    for (a, b) in pairs:
        M = S[(int(a), int(b))]
        M.sort_indices()
        rps.append(M.indptr.astype(np.int32))
        cols.append(M.indices.astype(np.int32))
        vals.append(M.data.astype(np.float32))
        rb.append(rb[-1] + int(L[a]) + 1)
        nb.append(nb[-1] + M.nnz)
    c = _Csr()
    c.pair_row_base = torch.tensor(rb, dtype=torch.int64, device=dev)
    c.pair_nnz_base = torch.tensor(nb, dtype=torch.int64, device=dev)
    c.row_ptr = torch.from_numpy(np.concatenate(rps)).to(dev)
    c.col_idx = torch.from_numpy(np.concatenate(cols + [np.zeros(1, np.int32)])).to(dev)
    c.val = torch.from_numpy(np.concatenate(vals + [np.zeros(1, np.float32)])).to(dev)
    return c, nb[-1]


def _compare(res, ref, cnt, pairs, fam, tau):
    rb = res.pair_row_base.cpu().numpy()
    nb = res.pair_nnz_base.cpu().numpy()
    rp_all, col_all, val_all = res.row_ptr.cpu().numpy(), res.col_idx.cpu().numpy(), res.val.cpu().numpy()
    relax = res.relaxations.cpu().numpy()
    L = fam.lengths
    worst = 0.0
    for p, (a, b) in enumerate(pairs):
        n, m = int(L[a]), int(L[b])
        rp = rp_all[rb[p]:rb[p] + n + 1]
        col, val = col_all[nb[p]:nb[p + 1]], val_all[nb[p]:nb[p + 1]]
        assert relax[p] == cnt[(int(a), int(b))], f"pair {p}: relaxations {relax[p]} vs {cnt[(int(a), int(b))]}"
        assert rp[0] == 0 and rp[-1] == len(col) and (np.diff(rp) >= 0).all()
        rows = np.repeat(np.arange(n), np.diff(rp))
        for i in np.nonzero(np.diff(rp) > 1)[0]:
            assert (np.diff(col[rp[i]:rp[i + 1]]) > 0).all(), f"pair {p} row {i}: columns not ascending"
        R = ref[(int(a), int(b))]
        Rd = R.toarray()
        got = np.zeros((n, m), dtype=bool)
        got[rows, col] = True
        # the oracle's un-thresholded relaxed values are needed for the band: recompute them with tau = 0 on demand
        must = Rd >= tau + BAND
        assert got[must].all(), f"pair {p}: {(must & ~got).sum()} relaxed entries >= tau + band missing"
        extra = got & (Rd == 0.0)
        if extra.any():
            _check_extra(p, extra, val, rows, col, tau)
        both = got & (Rd > 0.0)
        sel = both[rows, col]
        if sel.any():
            err = np.abs(val[sel] - Rd[rows[sel], col[sel]]).max()
            assert err <= S_ATOL, f"pair {p}: relaxed value error {err:.3e}"
            worst = max(worst, err)
    return worst


def _check_extra(p, extra, val, rows, col, tau):
    """Entries the kernel kept (so its value is >= tau) and the oracle dropped (its value is < tau): allowed only
    within the band above the threshold."""
    v = val[extra[rows, col]]
    assert (v < tau + BAND).all(), f"pair {p}: {int((v >= tau + BAND).sum())} entries kept that the oracle dropped"


def _run_case(fam, pairs, prm, T, f="max", h=3.0, passes=1, tau3=None):
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    S, td = _oracle_stage1(fam, pairs, prm)
    d_offs = torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev)
    d_pairs = torch.from_numpy(np.ascontiguousarray(pairs, dtype=np.int32)).to(dev)
    d_td = torch.from_numpy(np.ascontiguousarray(td, dtype=np.int32)).to(dev)
    csr, nnz = _upload(S, pairs, fam, dev)
    fsel = {"max": oc.SEL_MAX, "min": oc.SEL_MIN, "sum": oc.SEL_SUM}[f]
    worst = 0.0
    tau3 = prm.threshold if tau3 is None else tau3   # stage III's own threshold (normally stage I's)
    for it in range(passes):
        ref, cnt = oc.transform(S, fam.k, td, T=T, f=fsel, h=h, max_relax=200, tau=tau3)
        res = qp.consistency(d_offs, fam.k, d_pairs, csr, d_td, h_offsets=fam.offsets, h_pairs=pairs, nnz=nnz, T=T, f=f,
                             h=h, max_relax=200, threshold=tau3)
        worst = max(worst, _compare(res, ref, cnt, pairs, fam, tau3))
        if it + 1 < passes:
            # second transformation (k < 50): both sides continue from the ORACLE's first result
            S = {key: oc.from_csr(M.indptr, M.indices, M.data.astype(np.float32).astype(np.float64), *M.shape)
                 for key, M in ref.items()}
            csr, nnz = _upload(S, pairs, fam, dev)
    return worst, sum(cnt.values())


@pytest.mark.parametrize("T,f", [(5, "max"), (9, "max"), (200, "max"), (0, "max"), (12, "sum"), (5, "min")])
def test_cfg0_all_pairs(default_params, T, f):
    """configs[0] (8 proteins): every selection function, no / some / all sequences selected, two transformations
    (k < 50)."""
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    worst, nrel = _run_case(fam, pairs, default_params, T, f, passes=_qp().consistency_passes(fam.k))
    print(f"cfg0 T={T} f={f}: {nrel} relaxations, worst |dS'| {worst:.2e}")


@pytest.mark.parametrize("T", [0, 5, 200])
def test_threshold_above_stage_one_cuts_unrelaxed_pairs_too(default_params, T):
    """A stage-III threshold (0.05) above the one the input was cut at (0.01): include/qp.h drops relaxed values below
    it, and the oracle's relax_pair does so whether or not any z was selected -- so the pairs with |sel| = 0 (all of
    them at T = 0, some at T = 5) lose their small entries as well instead of being copied through unchanged."""
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    worst, nrel = _run_case(fam, pairs, default_params, T, tau3=0.05)
    assert (nrel == 0) == (T == 0)
    print(f"cfg0 T={T} tau3=0.05: {nrel} relaxations, worst |dS'| {worst:.2e}")


def test_cfg1_all_pairs(default_params):
    """configs[1] (50 sequences, 1,225 pairs): T = 25 selects subtrees of up to 13 leaves; 1 transformation (k >= 50)."""
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    assert _qp().consistency_passes(fam.k) == 1
    worst, nrel = _run_case(fam, pairs, default_params, T=25)
    assert nrel > 0
    print(f"cfg1 T=25: {nrel} relaxations, worst |dS'| {worst:.2e}")
    worst, nrel = _run_case(fam, pairs, default_params, T=200)      # every z selected: 48 relaxations per pair
    assert nrel == len(pairs) * (fam.k - 2)
    print(f"cfg1 T=200: {nrel} relaxations, worst |dS'| {worst:.2e}")


def test_ragged_orientations_and_missing_pairs(default_params):
    """Pairs listed in either orientation, some pairs absent (never relaxed over), very short and skewed sequences,
    rows with more than 32 stored cells (low threshold), more candidates than one selection block."""
    rng = np.random.default_rng(21)
    q = inputs.background()
    root = rng.choice(20, size=300, p=q).astype(np.uint8)
    seqs = []
    for L in (1, 2, 40, 300, 120, 77, 33, 250, 64, 65):
        s = root[:L].copy()
        hit = rng.random(L) < 0.3
        s[hit] = rng.choice(20, size=int(hit.sum()), p=q)
        seqs.append(s)
    fam = inputs.pack(seqs)
    pairs = inputs.all_pairs(fam.k)
    keep = rng.random(len(pairs)) < 0.85
    pairs = pairs[keep]
    flip = rng.random(len(pairs)) < 0.5
    pairs[flip] = pairs[flip][:, ::-1]
    prm = inputs.Params(hmm=default_params.hmm, pf=default_params.pf, threshold=0.0005)   # > 32 cells in many rows
    worst, nrel = _run_case(fam, np.ascontiguousarray(pairs), prm, T=200)
    assert nrel > 0
    print(f"ragged: {nrel} relaxations, worst |dS'| {worst:.2e}")


def test_many_sequences_selection_blocks_and_list_flush(default_params):
    """k = 300 short sequences: the candidates span two selection blocks of 256, and with every z selected the three
    pairs among sequences 0, 1, 2 are relaxed over 297 sequences each -- more than the shared-memory list holds at
    once, so the partial sums travel through the staging area between two flushes."""
    rng = np.random.default_rng(22)
    q = inputs.background()
    root = rng.choice(20, size=14, p=q).astype(np.uint8)
    seqs = []
    for s in range(300):
        L = int(rng.integers(8, 15))
        t = root[:L].copy()
        hit = rng.random(L) < 0.25
        t[hit] = rng.choice(20, size=int(hit.sum()), p=q)
        seqs.append(t)
    fam = inputs.pack(seqs)
    pairs = np.array([[a, b] for a in range(3) for b in range(a + 1, 300)], dtype=np.int32)
    worst, nrel = _run_case(fam, pairs, default_params, T=10 ** 6)
    assert nrel >= 3 * 297
    print(f"k=300: {nrel} relaxations, worst |dS'| {worst:.2e}")


def test_chain_stage1_tree_consistency_on_the_gpu(default_params):
    """The three stages chained on the device (qp_posteriors -> qp_guide_tree -> qp_consistency) on configs[1]: the
    call accepts the outputs of the earlier stages as they are, and the result agrees with the oracle chain wherever
    the stage-I patterns agree (stage-I band flips aside)."""
    import torch
    qp = _qp()
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    res1 = qp.run_family(fam, pairs, default_params)
    tree = qp.guide_tree(res1.dist)
    dev = res1.dist.device
    d_offs = torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev)
    d_pairs = torch.from_numpy(pairs).to(dev)
    res3 = qp.consistency(d_offs, fam.k, d_pairs, res1, tree.treedist, h_offsets=fam.offsets, h_pairs=pairs, T=25,
                          threshold=default_params.threshold)
    S, td = _oracle_stage1(fam, pairs, default_params)
    assert np.array_equal(td, tree.treedist.cpu().numpy())
    ref, cnt = oc.transform(S, fam.k, td, T=25, tau=default_params.threshold)
    assert np.array_equal(res3.relaxations.cpu().numpy(), np.array([cnt[(int(a), int(b))] for a, b in pairs]))
    nb = res3.pair_nnz_base.cpu().numpy()
    ref_nnz = np.array([ref[(int(a), int(b))].nnz for a, b in pairs])
    assert np.abs(np.diff(nb) - ref_nnz).sum() <= 0.002 * ref_nnz.sum() + 5     # only threshold-band cells may differ
    p = int(np.argmax(list(cnt.values())))
    rp, col, val = res3.csr(p)
    a, b = pairs[p]
    Rd = ref[(int(a), int(b))].toarray()
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    both = Rd[rows, col] > 0
    assert both.mean() > 0.99 and np.abs(val[both] - Rd[rows[both], col[both]]).max() <= 1e-4


def test_error_paths_and_empty_input(default_params):
    """qp_consistency argument and device-detected errors: bad pair, undersized workspace, undersized output, an empty
    pair list; and qp_shutdown between calls (the library re-creates its streams)."""
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    S, td = _oracle_stage1(fam, pairs, default_params)
    d_offs = torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev)
    d_pairs = torch.from_numpy(pairs).to(dev)
    d_td = torch.from_numpy(np.ascontiguousarray(td, dtype=np.int32)).to(dev)
    csr, nnz = _upload(S, pairs, fam, dev)
    kw = dict(h_offsets=fam.offsets, h_pairs=pairs, nnz=nnz, T=9, threshold=default_params.threshold)
    ok = qp.consistency(d_offs, fam.k, d_pairs, csr, d_td, **kw)
    assert ok.code == 0
    qp.shutdown()                                           # streams and events of this thread are released ...
    again = qp.consistency(d_offs, fam.k, d_pairs, csr, d_td, **kw)
    assert torch.equal(ok.val[:int(ok.pair_nnz_base[-1])], again.val[:int(again.pair_nnz_base[-1])])
    res1 = qp.run_family(fam, pairs, default_params)        # ... and re-created by the next stage-I call
    assert res1.code == 0
    # a pair that lists a sequence with itself: host query and device check
    bad = pairs.copy()
    bad[3] = (2, 2)
    with pytest.raises(qp.QpError) as ei:
        qp.consistency(d_offs, fam.k, torch.from_numpy(bad).to(dev), csr, d_td, **dict(kw, h_pairs=bad))
    assert ei.value.code == qp.ERR["BAD_PAIR"]
    # workspace too small
    small = torch.empty(1 << 16, dtype=torch.uint8, device=dev)
    with pytest.raises(qp.QpError) as ei:
        qp.consistency(d_offs, fam.k, d_pairs, csr, d_td, workspace=small, **kw)
    assert ei.value.code == qp.ERR["WORKSPACE_TOO_SMALL"]
    # an entry count smaller than what the matrices hold is caught for every pair, also for the pairs that are too far
    # apart to be a factor of anything (T = 0: nothing is selected, none of the copies is ever built)
    for T in (9, 0):
        with pytest.raises(qp.QpError) as ei:
            qp.consistency(d_offs, fam.k, d_pairs, csr, d_td, **dict(kw, nnz=nnz - 1, T=T))
        assert ei.value.code == qp.ERR["NNZ_CAPACITY"]
    # empty pair list
    none = np.zeros((0, 2), np.int32)
    r0 = qp.consistency(d_offs, fam.k, torch.from_numpy(none).to(dev), csr, d_td, **dict(kw, h_pairs=none, nnz=0))
    assert r0.code == 0 and int(r0.pair_nnz_base[0].item()) == 0


def test_fuzz_random_distance_matrices_selection_functions_and_amplification(default_params):
    """Seeded fuzz: ragged families (lengths 1..260, 4..14 sequences, some pairs missing, either orientation), distance
    matrices that are NOT tree distances (random symmetric integers), random T, f in {max, min, sum}, h in [1, 5],
    relaxation caps 1..11, thresholds 0.0005 .. 0.05 -- element by element against the oracle."""
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    total = 0
    for seed in range(1, 13):
        rng = np.random.default_rng(5000 + seed)
        q = inputs.background()
        k = int(rng.integers(4, 15))
        root = rng.choice(20, size=260, p=q).astype(np.uint8)
        seqs = []
        for _ in range(k):
            L = int(np.exp(rng.uniform(np.log(1), np.log(260))))
            s = root[:L].copy()
            hit = rng.random(L) < rng.uniform(0.05, 0.5)
            s[hit] = rng.choice(20, size=int(hit.sum()), p=q)
            seqs.append(s)
        fam = inputs.pack(seqs)
        pairs = inputs.all_pairs(fam.k)
        pairs = pairs[rng.random(len(pairs)) < rng.uniform(0.6, 1.0)]
        if len(pairs) == 0:
            continue
        flip = rng.random(len(pairs)) < 0.5
        pairs[flip] = pairs[flip][:, ::-1]
        pairs = np.ascontiguousarray(pairs)
        prm = inputs.Params(hmm=default_params.hmm, pf=default_params.pf, threshold=float(rng.choice([0.0005, 0.01, 0.05])))
        S, _ = _oracle_stage1(fam, pairs, prm)
        td = rng.integers(1, 30, size=(k, k))
        td = np.minimum(td, td.T)
        np.fill_diagonal(td, 1)
        T, f = int(rng.integers(0, 40)), str(rng.choice(["max", "min", "sum"]))
        h, mr = float(rng.uniform(1.0, 5.0)), int(rng.integers(1, 12))
        fsel = {"max": oc.SEL_MAX, "min": oc.SEL_MIN, "sum": oc.SEL_SUM}[f]
        ref, cnt = oc.transform(S, fam.k, td, T=T, f=fsel, h=h, max_relax=mr, tau=prm.threshold)
        d_offs = torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev)
        d_pairs = torch.from_numpy(pairs).to(dev)
        d_td = torch.from_numpy(np.ascontiguousarray(td, dtype=np.int32)).to(dev)
        csr, nnz = _upload(S, pairs, fam, dev)
        res = qp.consistency(d_offs, fam.k, d_pairs, csr, d_td, h_offsets=fam.offsets, h_pairs=pairs, nnz=nnz, T=T, f=f, h=h,
                             max_relax=mr, threshold=prm.threshold)
        _compare(res, ref, cnt, pairs, fam, prm.threshold)
        total += sum(cnt.values())
    assert total > 500
