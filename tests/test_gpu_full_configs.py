"""GPU parity at BASELINE.json's full sizes (configs[2], [3], [4]) in the launch configuration bench.py times:
device-resident inputs, production kernels (CSR + distance, fp32 with the fp64 distance re-evaluation), one call
over ALL pairs. The oracle cannot do 6e10 cells in a test, so
  * a seeded sample of pairs (plus the largest, smallest and most skewed ones) is compared with the oracle
    one by one: CSR pattern/values and distance, tolerances of BASELINE.json (tests/parity.py);
  * properties that hold at any size are checked on ALL pairs: distances symmetric and in [0,1], prefix arrays
    consistent, nnz per row <= min(m, floor(2/tau)) (SURVEY.md 8(c) pin 7), values in [tau, 1].
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import qp_oracle as orc
from paper_1512_07437_b200 import inputs
from tests import parity


def _run_full(cfg, prm):
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1512_07437_b200 import qp
    fam = inputs.config_family(cfg)
    pairs = inputs.all_pairs(fam.k)
    res = qp.run_family(fam, pairs, prm, precision="fp32", beta_guess=0.05)
    torch.cuda.synchronize()
    assert int(res.status[0].item()) == 0
    return fam, pairs, res


def _sample(fam, pairs, k, seed):
    L = fam.lengths
    n, m = L[pairs[:, 0]].astype(np.int64), L[pairs[:, 1]].astype(np.int64)
    cells = n * m
    pick = set(np.random.default_rng(seed).choice(len(pairs), size=k, replace=False).tolist())
    pick |= {int(np.argmax(cells)), int(np.argmin(cells)), int(np.argmax(n - m)), int(np.argmax(m - n))}
    return np.array(sorted(pick))


def _check_sample(fam, pairs, res, prm, idx):
    sub = np.ascontiguousarray(pairs[idx])
    run = orc.Run(prm, fam, sub, keep_dense=True)
    D = res.dist.cpu().numpy()
    worst_p = worst_d = 0.0
    for q, p in enumerate(idx):
        a, b = pairs[p]
        rp, col, val = res.csr(int(p))
        e = parity.check_pair(run.dense(q), run.dist[q], None, prm.threshold, rp, col, val, float(D[a, b]))
        worst_p, worst_d = max(worst_p, e[0]), max(worst_d, e[1])
    return worst_p, worst_d


def _check_all(fam, pairs, res, prm):
    import torch
    L = torch.from_numpy(fam.lengths.astype(np.int64)).cuda()
    pr = torch.from_numpy(pairs.astype(np.int64)).cuda()
    n, m = L[pr[:, 0]], L[pr[:, 1]]
    P = len(pairs)
    D = res.dist
    assert torch.equal(D, D.t()), "distance matrix not symmetric"
    d = D[pr[:, 0], pr[:, 1]]
    assert bool((d >= 0).all()) and bool((d <= 1).all()) and bool(torch.isfinite(d).all())
    rb, nb = res.pair_row_base, res.pair_nnz_base
    assert torch.equal(rb[1:] - rb[:-1], n + 1), "pair_row_base is not the prefix of n+1"
    assert int(nb[0].item()) == 0 and bool((nb[1:] >= nb[:-1]).all())
    rp = res.row_ptr[: int(rb[-1].item())].to(torch.int64)
    first, lastr = rb[:-1], rb[1:] - 1
    assert bool((rp[first] == 0).all()), "row_ptr[0] != 0"
    assert torch.equal(rp[lastr], nb[1:] - nb[:-1]), "row_ptr[n] != nnz of the pair"
    dr = rp[1:] - rp[:-1]
    inner = torch.ones_like(dr, dtype=torch.bool)
    inner[lastr[:-1]] = False                      # position of the jump from one pair's row_ptr to the next one's
    cap = int(2.0 / prm.threshold)
    assert bool((dr[inner] >= 0).all()), "row_ptr not monotone"
    assert int(dr[inner].max().item()) <= cap, "more than floor(2/tau) entries in a row"
    nnz = int(nb[-1].item())
    tau = np.float32(prm.threshold)
    step = 1 << 28
    for lo in range(0, nnz, step):
        v = res.val[lo:min(nnz, lo + step)]
        c = res.col_idx[lo:min(nnz, lo + step)]
        assert float(v.min().item()) >= tau and float(v.max().item()) <= 1.0 + 1e-5
        assert int(c.min().item()) >= 0
    # columns < m: per pair maximum via a segmented check on a strided subset of pairs (all pairs for small configs)
    sel = np.arange(0, P, max(1, P // 2000))
    nbh = nb.cpu().numpy()
    mh = m.cpu().numpy()
    for p in sel:
        if nbh[p + 1] > nbh[p]:
            assert int(res.col_idx[nbh[p]:nbh[p + 1]].max().item()) < mh[p]
    return nnz


@pytest.mark.parametrize("cfg,k_sample", [(2, 48), (4, 40), (3, 64)])
def test_full_config_sampled_parity_and_invariants(default_params, cfg, k_sample):
    fam, pairs, res = _run_full(cfg, default_params)
    nnz = _check_all(fam, pairs, res, default_params)
    idx = _sample(fam, pairs, k_sample, seed=7437100 + cfg)
    wp, wd = _check_sample(fam, pairs, res, default_params, idx)
    cells = int((fam.lengths[pairs[:, 0]].astype(np.int64) * fam.lengths[pairs[:, 1]]).sum())
    print(f"cfg{cfg}: {len(pairs)} pairs, {cells:.3e} cells, nnz {nnz} (beta {nnz / cells:.4f}); "
          f"{len(idx)} sampled pairs: worst |dP| {wp:.2e}, worst rel d {wd:.2e}")
