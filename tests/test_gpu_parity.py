"""GPU parity: CUDA path (through the C ABI, libqp.so) vs the fp64 oracle, element by element, same seeded inputs.

Tolerances are BASELINE.json's: dense posteriors max abs <= 1e-4, distances rel <= 1e-5, sparse pattern identical
except entries within 1e-4 of the threshold. Run with -m gpu on the B200 box.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import qp_oracle as orc
from paper_1512_07437_b200 import inputs
from tests import parity


def _qp():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1512_07437_b200 import qp
    return qp


def _compare(fam, pairs, params, res, run, dense=True, logZ=True, p_atol=parity.P_ATOL, d_rtol=parity.D_RTOL,
             logz_rtol=2e-6):
    D = res.dist.cpu().numpy()
    dn = res.dense_P.cpu().numpy() if dense else None
    lz = res.logZ.cpu().numpy() if logZ else None
    rb = res.pair_row_base.cpu().numpy()
    nb = res.pair_nnz_base.cpu().numpy()
    rp_all, col_all, val_all = res.row_ptr.cpu().numpy(), res.col_idx.cpu().numpy(), res.val.cpu().numpy()
    L = fam.lengths
    worst = (0.0, 0.0)
    for p, (a, b) in enumerate(pairs):
        n, m = int(L[a]), int(L[b])
        assert rb[p + 1] - rb[p] == n + 1
        rp = rp_all[rb[p]:rb[p + 1]]
        col, val = col_all[nb[p]:nb[p + 1]], val_all[nb[p]:nb[p + 1]]
        assert D[a, b] == D[b, a]
        d = dn[res.dense_off[p]:res.dense_off[p + 1]].reshape(n, m) if dense else None
        e = parity.check_pair(run.dense(p), run.dist[p], run.logZ(p), params.threshold, rp, col, val, float(D[a, b]),
                              dense=d, logZ=lz[p] if logZ else None, p_atol=p_atol, d_rtol=d_rtol,
                              logz_rtol=logz_rtol)
        worst = (max(worst[0], e[0]), max(worst[1], e[1]))
    return worst


def test_cfg0_fp64_all_pairs(default_params):
    """configs[0]: 8 proteins, lengths 60-100, all 28 pairs, fp64 posteriors."""
    qp = _qp()
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, precision="fp64", want_dense=True, want_logZ=True)
    worst = _compare(fam, pairs, default_params, res, run, p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11)
    assert worst[0] <= 1e-7
    # fp64 mode: the CSR pattern must be exactly the oracle's unless an entry is within 1e-7 of tau
    nb = res.pair_nnz_base.cpu().numpy()
    assert int(nb[-1]) == int(run.nnz.sum())


def test_cfg0_fp32_all_pairs(default_params):
    qp = _qp()
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, precision="fp32", want_dense=True, want_logZ=True)
    _compare(fam, pairs, default_params, res, run)
    assert int(res.status[3].item()) > 0      # cfg0 has near-identical pairs: the fp64 distance pass ran


def test_cfg1_fp32_all_pairs(default_params):
    """configs[1]: 50 sequences, mean length 250, all 1,225 pairs, fp32 GPU vs fp64 oracle."""
    qp = _qp()
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, precision="fp32", want_dense=True, want_logZ=True)
    worst = _compare(fam, pairs, default_params, res, run)
    print("cfg1 worst |dP| %.3e, worst rel d %.3e" % worst)


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_edge_lengths_and_ragged_tiles(default_params, precision):
    """length-1 and length-2 sequences, stripe-boundary lengths (63/64/65 ...), rows >> cols and cols >> rows."""
    qp = _qp()
    rng = np.random.default_rng(3)
    lens = [1, 1, 2, 3, 31, 32, 33, 63, 64, 65, 127, 128, 129, 255, 256, 257, 300, 511, 513, 40]
    fam = inputs.pack([rng.integers(0, 20, size=n).astype(np.uint8) for n in lens])
    pairs = inputs.all_pairs(fam.k)
    pairs = np.concatenate([pairs, pairs[::7, ::-1]])   # some pairs in both orientations
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, precision=precision, want_dense=True, want_logZ=True)
    tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else {}
    _compare(fam, pairs, default_params, res, run, **tol)


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_long_skewed_pairs_split_classes(default_params, precision):
    """configs[4]-style skew: pairs wider than one packed block go to the split classes (the warps of a CTA share
    the pair). 700 x 900 / 900 x 700 (3-4 blocks), 20 x 1500 and 1500 x 20, and 2500 columns = more blocks than
    warps (two passes, boundary column through the scratch slot)."""
    qp = _qp()
    rng = np.random.default_rng(4)
    q = inputs.background()
    base = rng.choice(20, size=900, p=q).astype(np.uint8)
    mut = base.copy()
    hit = rng.random(900) < 0.3
    mut[hit] = rng.choice(20, size=int(hit.sum()), p=q)
    fam = inputs.pack([base, mut[100:800], rng.integers(0, 20, size=20).astype(np.uint8),
                       rng.integers(0, 20, size=1500).astype(np.uint8), rng.choice(20, size=2500, p=q).astype(np.uint8),
                       rng.choice(20, size=45, p=q).astype(np.uint8)])
    # [3, 1] and [3, 0]: 1500 rows x 701 / 901 columns, too many cells for the two-block packed classes -> split C = 8
    pairs = np.array([[0, 1], [1, 0], [2, 3], [3, 2], [0, 3], [2, 1], [5, 4], [4, 5], [1, 4], [3, 1], [3, 0]], dtype=np.int32)
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, precision=precision, want_dense=True, want_logZ=True)
    tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else {}
    _compare(fam, pairs, default_params, res, run, **tol)


def test_near_identical_long_pairs_refined(default_params):
    """near-identical pairs (d < 0.25) of lengths 300 / 600 / 1100: the fp64 distance re-evaluation runs in the split
    fp64 classes (2,8), (4,8), (8,8)."""
    qp = _qp()
    rng = np.random.default_rng(8)
    q = inputs.background()
    seqs = []
    for L in (300, 600, 1100):
        a = rng.choice(20, size=L, p=q).astype(np.uint8)
        b = a.copy()
        hit = rng.random(L) < 0.05
        b[hit] = rng.choice(20, size=int(hit.sum()), p=q)
        seqs += [a, np.delete(b, slice(L // 2, L // 2 + 3))]
    fam = inputs.pack(seqs)
    pairs = np.array([[0, 1], [1, 0], [2, 3], [3, 2], [4, 5], [5, 4]], dtype=np.int32)
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, precision="fp32", want_dense=True, want_logZ=True)
    _compare(fam, pairs, default_params, res, run)
    assert int(res.status[3].item()) == len(pairs)
    assert float(run.dist.max()) < 0.25


def test_generic_models_g1_hmm_g2_pf():
    qp = _qp()
    rng = np.random.default_rng(5)
    prm = inputs.Params(hmm=inputs.random_model(rng, 1, 20), pf=inputs.random_model(rng, 2, 20), threshold=0.02)
    fam = inputs.random_family(rng, 6, 30, 140)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    for precision in ("fp32", "fp64"):
        res = qp.run_family(fam, pairs, prm, precision=precision, want_dense=True, want_logZ=True)
        tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else {}
        _compare(fam, pairs, prm, res, run, **tol)


def _pf_two_gap_states():
    """The default partition function with a second, long-gap insert-state pair (G = 2): dearer to open, cheaper to
    extend. Parameter values only (inputs), scaled by the default temperature 3."""
    pf, T = inputs.default_pf(), 3.0
    return inputs.Model(n_ins=2, alphabet=pf.alphabet, log_match=pf.log_match, log_ins=pf.log_ins, t_MM=0.0,
                        t_MI=(pf.t_MI[0], -16.0 / T), t_II=(pf.t_II[0], -0.4 / T), t_IM=(0.0, 0.0), init_M=0.0,
                        init_I=(pf.init_I[0], -16.0 / T), end_M=0.0, end_I=(0.0, 0.0))


def test_g2_partition_function_split_classes_and_distance_pass(default_params):
    """A partition function with TWO insert-state pairs through the fp32 SPLIT classes (launch_pair<float,2,C,*,4>,
    C = 8, 12, 16: columns 700 / 1300 / 2000, and 2600 = more blocks than warps), once with the test outputs
    (kModeFull) and once as the production instances (kModeCsr: no dense_P, no logZ), plus a near-identical pair so
    that the fp64 distance-only kernels run with GP = 2 (launch_pair<double,2,C,kModeDist,8>)."""
    qp = _qp()
    rng = np.random.default_rng(11)
    q = inputs.background()
    prm = inputs.Params(hmm=default_params.hmm, pf=_pf_two_gap_states(), threshold=0.01)
    seqs = [rng.choice(20, size=L, p=q).astype(np.uint8) for L in (700, 1300, 2000, 2600, 45)]
    a = rng.choice(20, size=800, p=q).astype(np.uint8)
    b = a.copy()
    hit = rng.random(800) < 0.04
    b[hit] = rng.choice(20, size=int(hit.sum()), p=q)
    seqs += [a, np.delete(b, slice(400, 403))]
    c = seqs[1].copy()                       # a diverged copy of the 1300-residue sequence: real structure in a wide pair
    hit = rng.random(1300) < 0.5
    c[hit] = rng.choice(20, size=int(hit.sum()), p=q)
    seqs.append(c)
    fam = inputs.pack(seqs)
    pairs = np.array([[4, 0], [0, 4], [0, 1], [1, 2], [4, 3], [3, 4], [2, 0], [5, 6], [6, 5], [7, 1], [1, 7], [0, 3]],
                     dtype=np.int32)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    assert float(run.dist.min()) < 0.25
    full = qp.run_family(fam, pairs, prm, precision="fp32", want_dense=True, want_logZ=True)
    _compare(fam, pairs, prm, full, run)
    prod = qp.run_family(fam, pairs, prm, precision="fp32")
    _compare(fam, pairs, prm, prod, run, dense=False, logZ=False)
    assert int(full.status[3].item()) >= 2 and int(prod.status[3].item()) >= 2   # the fp64 distance pass ran (GP = 2)


def test_g2_partition_function_production_instances_packed(default_params):
    """launch_pair<float,2,C,kModeCsr,1> for every packed stripe width C = 2..16: column counts 40, 72, ... , 488 (one
    per width), G = 2 partition function, production outputs only (CSR + distance) against the oracle's dense matrix."""
    qp = _qp()
    rng = np.random.default_rng(12)
    q = inputs.background()
    prm = inputs.Params(hmm=default_params.hmm, pf=_pf_two_gap_states(), threshold=0.01)
    root = rng.choice(20, size=520, p=q).astype(np.uint8)
    seqs = [root[:260].copy()]
    for C in range(2, 17):                   # m + 1 <= 32 C and > 32 (C - 1): the narrowest class that holds it is C
        s = root[: 32 * C - 24].copy()
        hit = rng.random(len(s)) < 0.35
        s[hit] = rng.choice(20, size=int(hit.sum()), p=q)
        seqs.append(s)
    fam = inputs.pack(seqs)
    pairs = np.array([[0, j] for j in range(1, 16)] + [[j, j + 1] for j in range(1, 15)], dtype=np.int32)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, prm, precision="fp32")
    _compare(fam, pairs, prm, res, run, dense=False, logZ=False)


@pytest.mark.parametrize("g2", [False, True])
def test_two_block_packed_classes(default_params, g2):
    """launch_pair<float,GP,C,MODE|kModeMB,1>, C = 9..12: pairs of 513..768 columns and moderate size on ONE warp that
    runs the two column blocks one after the other. One column count per stripe width (64 C - 20 and the smallest that
    needs the class), both orientations of the block boundary exercised by related sequences; with the test outputs
    (kModeFull) and as the production instances (kModeCsr); GP = 1 and GP = 2."""
    qp = _qp()
    rng = np.random.default_rng(13)
    q = inputs.background()
    prm = inputs.Params(hmm=default_params.hmm, pf=_pf_two_gap_states() if g2 else default_params.pf, threshold=0.01)
    root = rng.choice(20, size=1010, p=q).astype(np.uint8)
    seqs = [root[:300].copy(), root[350:610].copy()]
    for C in range(9, 13):
        for L in (64 * C - 20, 64 * (C - 1) + 1 if C > 9 else 513):
            s = root[:L].copy()
            hit = rng.random(L) < 0.3
            s[hit] = rng.choice(20, size=int(hit.sum()), p=q)
            seqs.append(s)
    fam = inputs.pack(seqs)
    pairs = np.array([[j % 2, 2 + j] for j in range(8)], dtype=np.int32)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    full = qp.run_family(fam, pairs, prm, precision="fp32", want_dense=True, want_logZ=True)
    _compare(fam, pairs, prm, full, run)
    prod = qp.run_family(fam, pairs, prm, precision="fp32")
    _compare(fam, pairs, prm, prod, run, dense=False, logZ=False)


def test_nucleotide_mode_alphabet_4():
    """PAPER.md:69 nucleotide mode: alphabet 4 through the same kernels (synthetic 4-letter model, the HOXD/GTR
    tables are not in the container). Related sequences (12 % substitutions, a few indels), lengths 150-600."""
    qp = _qp()
    rng = np.random.default_rng(9)
    prm = inputs.nucleotide_params()
    q = inputs.background(4)
    root = rng.choice(4, size=600, p=q).astype(np.uint8)
    seqs = []
    for L in (600, 450, 300, 150, 520):
        s = root.copy()
        hit = rng.random(600) < 0.12
        s[hit] = rng.choice(4, size=int(hit.sum()), p=q)
        cut = int(rng.integers(0, 600 - L + 1))
        s = s[cut:cut + L]
        seqs.append(np.delete(s, slice(L // 3, L // 3 + int(rng.integers(1, 6)))))
    fam = inputs.pack(seqs)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    for precision in ("fp32", "fp64"):
        res = qp.run_family(fam, pairs, prm, precision=precision, want_dense=True, want_logZ=True)
        tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else {}
        _compare(fam, pairs, prm, res, run, **tol)
    # a residue code outside the 4-letter alphabet is an error
    bad = inputs.Family(seqs=fam.seqs.copy(), offsets=fam.offsets.copy())
    bad.seqs[3] = 4
    with pytest.raises(qp.QpError) as ei:
        qp.run_family(bad, pairs, prm)
    assert ei.value.code == qp.ERR["BAD_RESIDUE"]


def test_error_paths(default_params):
    qp = _qp()
    import torch
    rng = np.random.default_rng(6)
    fam = inputs.random_family(rng, 4, 20, 40)
    pairs = inputs.all_pairs(fam.k)
    # nnz capacity too small -> NNZ_CAPACITY and the required size in pair_nnz_base[P]
    run = orc.Run(default_params, fam, pairs)
    with pytest.raises(qp.QpError) as ei:
        qp.run_family(fam, pairs, default_params, nnz_capacity=3)
    assert ei.value.code == qp.ERR["NNZ_CAPACITY"]
    # bad residue
    bad = inputs.Family(seqs=fam.seqs.copy(), offsets=fam.offsets.copy())
    bad.seqs[5] = 25
    with pytest.raises(qp.QpError) as ei:
        qp.run_family(bad, pairs, default_params)
    assert ei.value.code == qp.ERR["BAD_RESIDUE"]
    # bytes far outside the 32 x 32 emission table (255, and ASCII letters passed by mistake): the documented error,
    # no out-of-range shared-memory access (the context stays usable: the next call below succeeds)
    for junk in (255, None):
        bad = inputs.Family(seqs=fam.seqs.copy(), offsets=fam.offsets.copy())
        if junk is None:
            bad.seqs[:] = np.frombuffer(b"ACDEFGHIKLMNPQRSTVWY", dtype=np.uint8)[bad.seqs % 20]
        else:
            bad.seqs[7] = junk
        with pytest.raises(qp.QpError) as ei:
            qp.run_family(bad, pairs, default_params)
        assert ei.value.code == qp.ERR["BAD_RESIDUE"]
        torch.cuda.synchronize()
    # empty pair list is fine
    res = qp.run_family(fam, np.zeros((0, 2), np.int32), default_params)
    assert res.code == 0 and int(res.pair_nnz_base[0].item()) == 0
    # required nnz is reported on overflow
    cp = qp.CParams(default_params)
    dev = torch.device("cuda:0")
    d_seqs = torch.from_numpy(fam.seqs).to(dev)
    d_offs = torch.from_numpy(fam.offsets).to(dev)
    d_pairs = torch.from_numpy(pairs).to(dev)
    L = fam.lengths
    ws = torch.empty(qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, 3), dtype=torch.uint8, device=dev)
    r = qp.posteriors(d_seqs, d_offs, fam.k, d_pairs, cp, ws, nnz_capacity=3,
                      h_rows_total=int((L[pairs[:, 0]] + 1).sum()), check=False)
    assert r.code == qp.ERR["NNZ_CAPACITY"] and int(r.pair_nnz_base[-1].item()) == int(run.nnz.sum())


def test_host_streamer_matches_single_call(default_params):
    """stream.HostStreamer (host buffers, pair batches, two in flight) returns the same CSR and distances as one call."""
    qp = _qp()
    import torch
    from paper_1512_07437_b200 import stream
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    ref = qp.run_family(fam, pairs, default_params)
    rb, nb = ref.pair_row_base.cpu().numpy(), ref.pair_nnz_base.cpu().numpy()
    rp, col, val = ref.row_ptr.cpu().numpy(), ref.col_idx.cpu().numpy(), ref.val.cpu().numpy()
    hs = stream.HostStreamer(fam, pairs, default_params, batch_cells=1.0e7)     # 8 batches
    assert len(hs.bounds) - 1 >= 5
    for rep in range(2):                                                        # the streamer is reusable
        seen = 0
        for b in hs.run():
            assert b.lo == seen
            seen = b.hi
            n0, n1 = nb[b.lo], nb[b.hi]
            assert np.array_equal(b.nnz_base.numpy() - b.nnz_base.numpy()[0], nb[b.lo:b.hi + 1] - n0)
            assert np.array_equal(b.row_ptr.numpy(), rp[rb[b.lo]:rb[b.hi]])
            assert np.array_equal(b.col.numpy(), col[n0:n1]) and np.array_equal(b.val.numpy(), val[n0:n1])
        assert seen == len(pairs)
        assert torch.equal(hs.dist, ref.dist.cpu())
    # a capacity guess that is far too small: the overflowing batches are re-run in a grown slot, same result
    hs = stream.HostStreamer(fam, pairs, default_params, batch_cells=2.0e7, beta_guess=0.004)
    got = [(b.lo, b.hi, b.col.numpy().copy(), b.val.numpy().copy()) for b in hs.run()]
    assert hs.retries >= 1
    for lo, hi, c, v in got:
        assert np.array_equal(c, col[nb[lo]:nb[hi]]) and np.array_equal(v, val[nb[lo]:nb[hi]])
    assert torch.equal(hs.dist, ref.dist.cpu())


def test_host_call_matches_single_call(default_params):
    """qp_posteriors_host (host buffers in, host buffers out, batching inside the C library) returns the same CSR and
    distances as one device-resident call: default workspace, a workspace so small that batches must shrink, and a
    density guess so low that batches overflow and are split."""
    qp = _qp()
    import torch
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    ref = qp.run_family(fam, pairs, default_params)
    nz = int(ref.pair_nnz_base[-1].item())
    want = dict(rb=ref.pair_row_base.cpu(), nb=ref.pair_nnz_base.cpu(), rp=ref.row_ptr.cpu(), col=ref.col_idx[:nz].cpu(),
                val=ref.val[:nz].cpu(), dist=ref.dist.cpu())

    def same(hc):
        assert hc.code == 0 and hc.nnz == nz
        assert torch.equal(hc.pair_row_base, want["rb"]) and torch.equal(hc.pair_nnz_base, want["nb"])
        assert torch.equal(hc.row_ptr[: len(want["rp"])], want["rp"])
        assert torch.equal(hc.col_idx[:nz], want["col"]) and torch.equal(hc.val[:nz], want["val"])
        assert torch.equal(hc.dist, want["dist"])
        assert hc.refined == int(ref.status[3].item())
        assert hc.d2h_bytes >= 8 * nz and hc.h2d_bytes >= fam.seqs.nbytes

    hc = qp.HostCall(fam, pairs, default_params)
    same(hc.run())
    same(hc.run())                                             # reusable
    small = qp.HostCall(fam, pairs, default_params, workspace_bytes=hc.ws.numel() // 6)
    same(small.run())
    assert small.batches > hc.batches
    dense = qp.HostCall(fam, pairs, default_params, beta_guess=0.004, nnz_capacity=nz + 16)
    same(dense.run())
    assert dense.batches > hc.batches                          # overflowing batches were split
    # the same with 16-bit columns: the narrowing kernel of an overflowing batch must stop at the slot's capacity (it
    # once walked on to the size the batch NEEDED and overwrote the slot's status word and workspace)
    dense16 = qp.HostCall(fam, pairs, default_params, beta_guess=0.004, nnz_capacity=nz + 16, compact_cols=True).run()
    assert dense16.code == 0 and dense16.nnz == nz and dense16.batches > hc.batches
    assert torch.equal(dense16.col_idx16[:nz].to(torch.int32), want["col"]) and torch.equal(dense16.val[:nz], want["val"])
    assert torch.equal(dense16.dist, want["dist"]) and torch.equal(dense16.pair_nnz_base, want["nb"])
    compact = qp.HostCall(fam, pairs, default_params, compact_cols=True).run()      # columns as uint16: 6 B / entry
    assert compact.code == 0 and compact.nnz == nz and compact.col_idx is None
    assert torch.equal(compact.col_idx16[:nz].to(torch.int32), want["col"]) and torch.equal(compact.val[:nz], want["val"])
    assert compact.d2h_bytes < hc.d2h_bytes - nz
    tight = qp.HostCall(fam, pairs, default_params, nnz_capacity=nz // 2)
    tight.run(check=False)
    assert tight.code == qp.ERR["NNZ_CAPACITY"] and int(tight.pair_nnz_base[len(pairs)].item()) == nz


def test_sharded_pair_list_on_the_gpu_matches_one_call(default_params):
    """SURVEY.md 8(e) on one device: the three shards that multi.ShardedFamily deals to a world of 3 ranks, run one
    after the other through qp_posteriors, give bit for bit the distances and the per-pair CSR of the unsharded call
    (the exchange itself -- a sum of matrices with disjoint supports -- is covered by tests/test_multi_gloo.py)."""
    qp = _qp()
    import torch
    from paper_1512_07437_b200 import multi
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    ref = qp.run_family(fam, pairs, default_params)
    rb, nb = ref.pair_row_base.cpu().numpy(), ref.pair_nnz_base.cpu().numpy()
    col, val = ref.col_idx.cpu().numpy(), ref.val.cpu().numpy()
    total = torch.zeros_like(ref.dist)
    seen = np.zeros(len(pairs), dtype=bool)
    for rank in range(3):
        sh = multi.ShardedFamily(fam.lengths, pairs, 3, rank)
        part = qp.run_family(fam, sh.pairs, default_params)
        total += sh.step(lambda _pairs: part.dist)          # no process group: the exchange is the identity
        pnb = part.pair_nnz_base.cpu().numpy()
        pcol, pval = part.col_idx.cpu().numpy(), part.val.cpu().numpy()
        for q, p in enumerate(sh.mine):
            assert not seen[p]
            seen[p] = True
            assert np.array_equal(pcol[pnb[q]:pnb[q + 1]], col[nb[p]:nb[p + 1]])
            assert np.array_equal(pval[pnb[q]:pnb[q + 1]], val[nb[p]:nb[p + 1]])
    assert seen.all() and torch.equal(total, ref.dist)


def test_fuzz_random_pairs_models_thresholds():
    """Seeded fuzz: random lengths (1..400, incl. very skewed pairs), random symmetric models with G in {1,2} for
    either automaton, alphabets 4 / 12 / 20 / 31, thresholds 0.001 .. 0.2, both precisions."""
    qp = _qp()
    rng = np.random.default_rng(20240607)
    for trial in range(6):
        A = int(rng.choice([4, 12, 20, 31]))
        gh, gp = int(rng.integers(1, 3)), int(rng.integers(1, 3))
        prm = inputs.Params(hmm=inputs.random_model(rng, gh, A), pf=inputs.random_model(rng, gp, A),
                            threshold=float(rng.choice([0.001, 0.01, 0.05, 0.2])))
        lens = [int(v) for v in rng.integers(1, 400, size=7)] + [1, 2]
        fam = inputs.pack([rng.integers(0, A, size=n).astype(np.uint8) for n in lens])
        pairs = inputs.all_pairs(fam.k)
        pairs = pairs[rng.permutation(len(pairs))[:20]]
        flip = rng.random(len(pairs)) < 0.5
        pairs[flip] = pairs[flip][:, ::-1]
        run = orc.Run(prm, fam, pairs, keep_dense=True)
        for precision in ("fp32", "fp64"):
            res = qp.run_family(fam, pairs, prm, precision=precision, want_dense=True, want_logZ=True)
            tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else dict(logz_rtol=5e-6)
            _compare(fam, pairs, prm, res, run, **tol)


def test_workspace_budget_gives_same_result(default_params):
    """A capped workspace (fewer scratch slots, pairs wait for a slot) changes the schedule, not the result."""
    qp = _qp()
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)
    full = qp.run_family(fam, pairs, default_params)
    cp = qp.CParams(default_params)
    cap = int(full.pair_nnz_base[-1].item()) + 16
    need = qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, cap)
    small = qp.run_family(fam, pairs, default_params, nnz_capacity=cap, budget=need // 6)
    assert qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, cap, budget=need // 6) <= need // 6
    for name in ("pair_nnz_base", "row_ptr", "dist"):
        assert (getattr(full, name).cpu().numpy()[: len(getattr(small, name))] == getattr(small, name).cpu().numpy()).all(), name
    nz = int(full.pair_nnz_base[-1].item())
    assert (full.col_idx[:nz] == small.col_idx[:nz]).all() and (full.val[:nz] == small.val[:nz]).all()


def test_memory_limited_mode_raises_threshold(default_params):
    """PAPER.md:73 memory-limited mode: the CSR capacity is the budget; the threshold is raised until the CSR fits and
    the result is exactly the posterior stage at the threshold that is reported back."""
    qp = _qp()
    import torch
    fam = inputs.config_family(1)
    pairs = inputs.all_pairs(fam.k)[:300]
    full = qp.run_family(fam, pairs, default_params)
    nnz_full = int(full.pair_nnz_base[-1].item())
    cap = nnz_full // 3
    dev = torch.device("cuda:0")
    cp = qp.CParams(default_params)
    L = fam.lengths
    ws = torch.empty(qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, cap), dtype=torch.uint8, device=dev)
    args = (torch.from_numpy(fam.seqs).to(dev), torch.from_numpy(fam.offsets).to(dev), fam.k, torch.from_numpy(pairs).to(dev), cp, ws)
    kw = dict(nnz_capacity=cap, h_rows_total=int((L[pairs[:, 0]] + 1).sum()))
    res = qp.posteriors(*args, budget_passes=8, **kw)
    assert res.code == 0 and res.passes == 2 and res.tau_used > default_params.threshold      # never more than two passes
    nnz = int(res.pair_nnz_base[-1].item())
    assert nnz <= cap
    # the threshold comes off the histogram of the first pass: a bin edge, the smallest one that fits, exactly
    tau, cnt = qp.last_tau_curve()
    assert tau[0] == np.float32(default_params.threshold) and cnt[0] == nnz_full and (np.diff(cnt) <= 0).all()
    b = int(np.nonzero(tau == res.tau_used)[0][0])
    assert cnt[b] == nnz and cnt[b - 1] > cap
    print(f"budget {cap} entries of {nnz_full}: tau {default_params.threshold} -> {res.tau_used:.4f} in {res.passes} passes, nnz {nnz}")
    prm = inputs.Params(hmm=default_params.hmm, pf=default_params.pf, threshold=res.tau_used)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    _compare(fam, pairs, prm, res, run, dense=False, logZ=False)
    assert abs(nnz - int(run.nnz.sum())) <= 0.001 * nnz + 5          # only threshold-band entries may differ
    # one pass is not enough: the capacity error comes back with the threshold that was tried last
    r1 = qp.posteriors(*args, budget_passes=1, check=False, **kw)
    assert r1.code == qp.ERR["NNZ_CAPACITY"] and r1.passes == 1 and int(r1.pair_nnz_base[-1].item()) == nnz_full


def test_call_can_be_captured_into_a_cuda_graph(default_params):
    """qp_posteriors only enqueues work (flags = 0: no host synchronisation, no allocation): the whole call, side streams
    included, can be captured into a CUDA graph and replayed; the replay writes bit for bit what the plain call wrote."""
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    L = fam.lengths
    n, m = L[pairs[:, 0]].astype(np.int64), L[pairs[:, 1]].astype(np.int64)
    cells, rows = int((n * m).sum()), int((n + 1).sum())
    d_seqs = torch.from_numpy(np.ascontiguousarray(fam.seqs)).to(dev)
    d_offs = torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev)
    d_pairs = torch.from_numpy(pairs).to(dev)
    cp = qp.CParams(default_params, flags=0)
    cap = int(0.2 * cells) + 1024
    ws = torch.empty(qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, cap), dtype=torch.uint8, device=dev)
    kw = dict(nnz_capacity=cap, h_rows_total=rows, check=False)
    ref = qp.posteriors(d_seqs, d_offs, fam.k, d_pairs, cp, ws, **kw)
    torch.cuda.synchronize()
    assert int(ref.status[0].item()) == 0
    want = [t.clone() for t in (ref.dist, ref.pair_nnz_base, ref.row_ptr, ref.col_idx, ref.val)]
    out = qp.alloc_outputs(dev, len(pairs), rows, cap, fam.k)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):   # warm-up on the capture stream (creates the library's side streams before the capture)
        qp.posteriors(d_seqs, d_offs, fam.k, d_pairs, cp, ws, reuse=out, stream=s, **kw)
    torch.cuda.current_stream().wait_stream(s)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        qp.posteriors(d_seqs, d_offs, fam.k, d_pairs, cp, ws, reuse=out, stream=s, **kw)
    for _ in range(2):
        for t in (out.dist, out.val, out.col_idx, out.row_ptr, out.pair_nnz_base, out.status):
            t.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert out.status.tolist()[0] == 0 and out.status.tolist()[3] == int(ref.status[3].item())
        nnz = int(want[1][-1].item())
        got = (out.dist, out.pair_nnz_base, out.row_ptr, out.col_idx, out.val)
        for a, b, name in zip(got, want, ("dist", "pair_nnz_base", "row_ptr", "col_idx", "val")):
            k = nnz if name in ("col_idx", "val") else b.numel()
            assert torch.equal(a[:k] if a.dim() == 1 else a, b[:k] if b.dim() == 1 else b), name


def test_rows_much_longer_than_columns_in_a_wide_stripe(default_params):
    """Unrelated sequences of 1029 / 1285 rows against 489 columns (class C = 16) under a random two-insert-state model:
    the path has to cross every 16-column stripe through long gaps, F peaks at one end of a stripe and B at the other,
    and the posterior scale exponent of qp_lane.h (PScale) reaches 65..96. Round 1 reported QP_ERR_RANGE here although
    every posterior is representable; now the call succeeds and matches the oracle in both precisions."""
    qp = _qp()
    rng = np.random.default_rng(6)
    A = int(rng.choice([4, 12, 20, 31]))
    gh, gp = int(rng.integers(1, 3)), int(rng.integers(1, 3))
    prm = inputs.Params(hmm=inputs.random_model(rng, gh, A), pf=inputs.random_model(rng, gp, A),
                        threshold=float(rng.choice([0.001, 0.01, 0.05, 0.2])))
    lens = [int(v) for v in rng.integers(1, 1300, size=7)] + [1, 2, 33]
    assert (A, gh, gp) == (12, 2, 2) and lens[2] == 489 and lens[3] == 1029 and lens[6] == 1285
    fam = inputs.pack([rng.integers(0, A, size=n).astype(np.uint8) for n in lens])
    pairs = np.array([[3, 2], [6, 2], [2, 3], [2, 6]], dtype=np.int32)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    for precision in ("fp32", "fp64"):
        res = qp.run_family(fam, pairs, prm, precision=precision, want_dense=True, want_logZ=True)
        tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else dict(logz_rtol=5e-6)
        _compare(fam, pairs, prm, res, run, **tol)
    res = qp.run_family(fam, pairs, prm)   # production instances
    _compare(fam, pairs, prm, res, run, dense=False, logZ=False)


@pytest.mark.parametrize("seed", [14, 15, 18, 19])
def test_fuzz_skewed_length_regimes(seed):
    """Seeded fuzz over length regimes the configs do not reach: a few very short sequences against 1 500..3 200 residues
    (every split class, several passes), and log-uniform lengths 2..2 500; random models (G in {1, 2} per automaton,
    alphabets 4..31), random thresholds; test instances and production instances, both precisions."""
    qp = _qp()
    rng = np.random.default_rng(seed)
    A = int(rng.choice([4, 12, 20, 31]))
    gh, gp = int(rng.integers(1, 3)), int(rng.integers(1, 3))
    prm = inputs.Params(hmm=inputs.random_model(rng, gh, A), pf=inputs.random_model(rng, gp, A),
                        threshold=float(rng.choice([0.001, 0.01, 0.05, 0.2])))
    if seed % 4 == 2:
        lens = [int(v) for v in rng.integers(1, 60, size=4)] + [int(v) for v in rng.integers(1500, 3200, size=3)] + [513, 769]
    else:
        lens = [int(v) for v in np.exp(rng.uniform(np.log(2), np.log(2500), size=9))]
    fam = inputs.pack([rng.integers(0, A, size=n).astype(np.uint8) for n in lens])
    pairs = inputs.all_pairs(fam.k)
    pairs = pairs[rng.permutation(len(pairs))[:24]]
    flip = rng.random(len(pairs)) < 0.5
    pairs[flip] = pairs[flip][:, ::-1]
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    for precision in ("fp32", "fp64"):
        tol = dict(p_atol=1e-7, d_rtol=1e-6, logz_rtol=1e-11) if precision == "fp64" else dict(logz_rtol=5e-6)
        res = qp.run_family(fam, pairs, prm, precision=precision, want_dense=True, want_logZ=True)
        _compare(fam, pairs, prm, res, run, **tol)
        res = qp.run_family(fam, pairs, prm, precision=precision)
        _compare(fam, pairs, prm, res, run, dense=False, logZ=False, **tol)


@pytest.mark.parametrize("seed", [2, 5, 7])
def test_fuzz_identical_and_near_identical_sequences(seed):
    """Identical sequences and copies with 1 % / 8 % substitutions and a short deletion, lengths 1..2 600 (log-uniform),
    protein and nucleotide models: every pair goes through the fp64 distance queue (all three fp64 classes); distances
    to relative 1e-5 against the oracle, posteriors to 1e-4."""
    qp = _qp()
    rng = np.random.default_rng(1000 + seed)
    nuc = seed % 5 == 0
    prm = inputs.nucleotide_params() if nuc else inputs.default_params()
    A = 4 if nuc else 20
    seqs = []
    for _ in range(4):
        n = int(np.exp(rng.uniform(np.log(1), np.log(2600))))
        base = rng.integers(0, A, size=max(n, 1)).astype(np.uint8)
        seqs.append(base)
        for rate in (0.0, 0.01, 0.08):
            s = base.copy()
            mut = rng.random(len(s)) < rate
            s[mut] = rng.integers(0, A, size=int(mut.sum()))
            if len(s) > 10 and rate > 0:
                cut = int(rng.integers(0, len(s) - 3))
                s = np.concatenate([s[:cut], s[cut + int(rng.integers(1, 3)):]])
            seqs.append(s.astype(np.uint8))
    fam = inputs.pack(seqs)
    pairs = np.array([(4 * g + a, 4 * g + b) if (a + b + seed) % 2 else (4 * g + b, 4 * g + a)
                      for g in range(4) for a in range(4) for b in range(a + 1, 4)], dtype=np.int32)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, prm, want_dense=True, want_logZ=True, beta_guess=0.3)
    _compare(fam, pairs, prm, res, run)
    assert int(res.status[3].item()) == len(pairs)          # every pair was re-evaluated in fp64
    res = qp.run_family(fam, pairs, prm, beta_guess=0.3)
    _compare(fam, pairs, prm, res, run, dense=False, logZ=False)


def test_maximum_sequence_length(default_params):
    """QP_MAX_LEN = 65 535 residues as rows and as columns (128 column blocks of the widest split class, 16 passes),
    against a medium and a short sequence, plus a 40 000-residue near copy (the fp64 distance queue at that length).
    fp32 at the usual tolerances; the fp64 mode at 1e-6 on P: at |ln Z| ~ 2e5 the ORACLE's log-space fp64 values have an
    absolute rounding error of 3e-11 per operation, which 65 535 rows accumulate to ~1e-7."""
    qp = _qp()
    rng = np.random.default_rng(77)
    q = inputs.background()
    big = rng.choice(20, size=65535, p=q).astype(np.uint8)
    mid = big[30000:30300].copy()
    hit = rng.random(300) < 0.3
    mid[hit] = rng.choice(20, size=int(hit.sum()), p=q)
    small = big[100:120].copy()
    near = big[:40000].copy()
    hit = rng.random(40000) < 0.02
    near[hit] = rng.choice(20, size=int(hit.sum()), p=q)
    tiny = big[5000:5005].copy()
    fam = inputs.pack([big, mid, small, near, tiny])
    # [4, 0]: 5 rows against 65 535 columns = 171 column blocks run by ONE warp (short rows: the multi-block class)
    pairs = np.array([[0, 1], [1, 0], [0, 2], [2, 0], [3, 1], [1, 3], [4, 0], [0, 4], [4, 3]], dtype=np.int32)
    run = orc.Run(default_params, fam, pairs, keep_dense=True)
    res = qp.run_family(fam, pairs, default_params, want_dense=True, want_logZ=True, beta_guess=0.02)
    _compare(fam, pairs, default_params, res, run, logz_rtol=5e-6)
    res = qp.run_family(fam, pairs, default_params, beta_guess=0.02)
    _compare(fam, pairs, default_params, res, run, dense=False, logZ=False)
    res = qp.run_family(fam, pairs, default_params, precision="fp64", beta_guess=0.02)
    _compare(fam, pairs, default_params, res, run, dense=False, logZ=False, p_atol=1e-6, d_rtol=1e-6)
    # one residue more is refused
    over = inputs.pack([np.zeros(65536, np.uint8), small])
    with pytest.raises(qp.QpError) as ei:
        qp.run_family(over, np.array([[0, 1]], dtype=np.int32), default_params)
    assert ei.value.code == qp.ERR["EMPTY_SEQUENCE"]


def test_concurrent_callers_threads_and_interleaved_streams(default_params):
    """The library keeps its side streams and events per host thread and device: four host threads calling at the same
    time, and one thread interleaving calls on two streams (separate workspaces, no synchronisation in between), all get
    bit for bit the results of calls made one after the other."""
    import threading
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    fams = [inputs.config_family(1), inputs.config_family(0), inputs.random_family(np.random.default_rng(3), 30, 50, 400)]
    refs = []
    for fam in fams:
        pairs = inputs.all_pairs(fam.k)
        r = qp.run_family(fam, pairs, default_params)
        nz = int(r.pair_nnz_base[-1].item())
        refs.append((pairs, r.dist.clone(), r.val[:nz].clone(), r.col_idx[:nz].clone(), r.pair_nnz_base.clone()))

    def same(r, ref):
        nz = int(ref[4][-1].item())
        return (int(r.status[0].item()) == 0 and torch.equal(r.dist, ref[1]) and torch.equal(r.val[:nz], ref[2]) and
                torch.equal(r.col_idx[:nz], ref[3]) and torch.equal(r.pair_nnz_base, ref[4]))

    outs = [[] for _ in range(4)]

    def worker(i):
        try:
            for _ in range(4):
                outs[i].append(same(qp.run_family(fams[i % 3], refs[i % 3][0], default_params), refs[i % 3]))
        except Exception as e:   # noqa: BLE001 -- reported through the assertion below
            outs[i].append(repr(e))

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(4)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert all(o == [True] * 4 for o in outs), outs

    def setup(fam, pairs):
        L = fam.lengths
        n, m = L[pairs[:, 0]].astype(np.int64), L[pairs[:, 1]].astype(np.int64)
        cp = qp.CParams(default_params, flags=0)
        cap = int(0.1 * int((n * m).sum())) + 4096
        ws = torch.empty(qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, cap), dtype=torch.uint8, device=dev)
        args = (torch.from_numpy(np.ascontiguousarray(fam.seqs)).to(dev),
                torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev), fam.k,
                torch.from_numpy(pairs).to(dev), cp, ws)
        return args, dict(nnz_capacity=cap, h_rows_total=int((n + 1).sum()), check=False)

    (a_args, a_kw), (b_args, b_kw) = setup(fams[0], refs[0][0]), setup(fams[2], refs[2][0])
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(4):
        ra = qp.posteriors(*a_args, stream=s1, **a_kw)
        rb = qp.posteriors(*b_args, stream=s2, **b_kw)
        ra = qp.posteriors(*a_args, stream=s1, reuse=ra, **a_kw)
        torch.cuda.synchronize()
        assert same(ra, refs[0]) and same(rb, refs[2])


@pytest.mark.timeout(600, method="thread")
def test_large_calls_in_flight_with_pollers_finish_and_agree(default_params):
    """Three configs[2]-sized calls (19 900 pairs each, every one wide enough to fill the GPU by itself), WITH the fp64
    pollers, enqueued back to back on three streams without any synchronisation in between, ten rounds: every call
    finishes and returns bit for bit what it returns alone. The pollers of one call wait for that call's fp32 kernels;
    with several calls in flight their CTAs could once have covered the SMs before those kernels were resident. They now
    claim only visible queue entries and leave after a bounded number of empty polls (csrc/qp_kernel.cuh), so progress
    does not depend on which CTAs the hardware places first."""
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    fam = inputs.config_family(2)
    pairs = inputs.all_pairs(fam.k)
    ref = qp.run_family(fam, pairs, default_params)
    nz = int(ref.pair_nnz_base[-1].item())
    assert int(ref.status[3].item()) > 0, "the family must send pairs through the fp64 queue for this test to mean anything"
    L = fam.lengths
    n, m = L[pairs[:, 0]].astype(np.int64), L[pairs[:, 1]].astype(np.int64)
    cp = qp.CParams(default_params, flags=0)   # pollers on (no QP_FLAG_NO_POLLERS), no synchronisation inside the call
    cap = nz + 4096
    d_seqs = torch.from_numpy(np.ascontiguousarray(fam.seqs)).to(dev)
    d_offs = torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev)
    d_pairs = torch.from_numpy(pairs).to(dev)
    wsb = qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, cap)
    wss = [torch.empty(wsb, dtype=torch.uint8, device=dev) for _ in range(3)]
    streams = [torch.cuda.Stream() for _ in range(3)]
    kw = dict(nnz_capacity=cap, h_rows_total=int((n + 1).sum()), check=False)
    res = [None] * 3
    torch.cuda.synchronize()
    for _ in range(10):
        for q in range(3):
            res[q] = qp.posteriors(d_seqs, d_offs, fam.k, d_pairs, cp, wss[q], stream=streams[q], reuse=res[q], **kw)
        torch.cuda.synchronize()
        for r in res:
            assert int(r.status[0].item()) == 0 and int(r.status[3].item()) == int(ref.status[3].item())
            assert torch.equal(r.dist, ref.dist) and torch.equal(r.pair_nnz_base, ref.pair_nnz_base)
            assert torch.equal(r.val[:nz], ref.val[:nz]) and torch.equal(r.col_idx[:nz], ref.col_idx[:nz])


@pytest.mark.parametrize("kind", ["random", "log_uniform", "near_identical"])
def test_minimum_workspace_is_enough(default_params, kind):
    """A workspace of EXACTLY the minimum that qp_workspace_bytes reports (one scratch slot per class) runs the call and
    gives bit for bit the results of a full-size workspace. (The slots of the fp64 pollers once came off the top
    regardless and left the fp32 classes short: QP_ERR_WORKSPACE_TOO_SMALL at the advertised minimum.)"""
    import torch
    qp = _qp()
    dev = torch.device("cuda:0")
    rng = np.random.default_rng({"random": 708, "log_uniform": 705, "near_identical": 702}[kind])
    if kind == "random":
        fam = inputs.random_family(rng, 12, 1, 300)
    elif kind == "log_uniform":
        fam = inputs.pack([rng.integers(0, 20, size=int(n)).astype(np.uint8)
                           for n in np.exp(rng.uniform(np.log(2), np.log(2500), size=8))])
    else:
        base = rng.integers(0, 20, size=900).astype(np.uint8)
        fam = inputs.pack([base] + [np.where(rng.random(900) < 0.03, rng.integers(0, 20, size=900), base).astype(np.uint8)
                                    for _ in range(6)])
    pairs = inputs.all_pairs(fam.k)
    ref = qp.run_family(fam, pairs, default_params, beta_guess=0.3)
    nz = int(ref.pair_nnz_base[-1].item())
    cp = qp.CParams(default_params)
    full = qp.workspace_bytes(fam.offsets, fam.k, pairs, cp, nz + 8)
    least = qp.min_workspace_bytes(fam.offsets, fam.k, pairs, cp, nz + 8)
    assert least < full
    L = fam.lengths
    args = (torch.from_numpy(np.ascontiguousarray(fam.seqs)).to(dev),
            torch.from_numpy(np.ascontiguousarray(fam.offsets, dtype=np.int64)).to(dev), fam.k, torch.from_numpy(pairs).to(dev), cp)
    for wsb in (least, (least + full) // 2):
        ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        res = qp.posteriors(*args, ws, nnz_capacity=nz + 8, h_rows_total=int((L[pairs[:, 0]] + 1).sum()), check=False)
        assert res.code == 0, (wsb, res.status.tolist())
        assert torch.equal(res.dist, ref.dist) and torch.equal(res.pair_nnz_base, ref.pair_nnz_base)
        assert torch.equal(res.val[:nz], ref.val[:nz]) and torch.equal(res.col_idx[:nz], ref.col_idx[:nz])
        assert int(res.status[3].item()) == int(ref.status[3].item())
