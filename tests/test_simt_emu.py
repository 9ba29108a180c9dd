"""CPU check of the CUDA path's lane arithmetic and wavefront logic (qp_lane.h) via lockstep emulation of a warp.

The GPU parity tests (-m gpu) are the parity tests proper; this exists so that the kernel logic (start/end
injection, block-floating-point renormalisation, multi-block boundary hand-over, MEA, CSR traversal order) is
exercised by the CPU suite on a box without a GPU. Expected values come from the oracle only.
"""
import numpy as np
import pytest

from oracle import qp_oracle as orc
from paper_1512_07437_b200 import inputs
from tests.simt_emu import emu


def _check(params, x, y, C, fp64=False, GP=None, p_tol=1e-4, d_rtol=1e-4, mask=7):
    ref = orc.pair(params, x, y)
    r = emu.run(params, x, y, C, fp64=fp64, GP=GP, mask=mask)
    assert r.code == 0
    assert np.abs(r.P - ref.P).max() <= p_tol
    assert r.dist == pytest.approx(ref.dist, rel=d_rtol, abs=1e-6)
    np.testing.assert_allclose(r.logZ, ref.logZ, rtol=2e-6 if not fp64 else 1e-11)
    # CSR: identical outside the +-1e-4 threshold band, rows/cols ascending
    tau = params.threshold
    must = ref.P >= tau + 1e-4
    may = ref.P >= tau - 1e-4
    got = np.zeros_like(must)
    got[r.rows, r.cols] = True
    assert (got[must]).all() and not (got & ~may).any()
    assert (np.diff(r.row_ptr) >= 0).all() and r.row_ptr[-1] == len(r.cols)
    for i in range(len(x)):
        c = r.cols[r.row_ptr[i]:r.row_ptr[i + 1]]
        assert (r.rows[r.row_ptr[i]:r.row_ptr[i + 1]] == i).all() and (np.diff(c) > 0).all()
    np.testing.assert_allclose(r.vals, ref.P[r.rows, r.cols], atol=p_tol)
    return r, ref


@pytest.mark.parametrize("n,m,C", [(1, 1, 2), (1, 2, 2), (2, 1, 2), (3, 63, 2), (40, 31, 2), (64, 65, 4), (90, 127, 4),
                                   (70, 255, 8), (33, 300, 10), (120, 100, 16), (50, 90, 3), (33, 270, 9)])
def test_emu_fp32_single_block(default_params, n, m, C):
    rng = np.random.default_rng(n * 1000 + m)
    q = inputs.background()
    x = rng.choice(20, size=n, p=q).astype(np.uint8)
    y = rng.choice(20, size=m, p=q).astype(np.uint8)
    _check(default_params, x, y, C)


@pytest.mark.parametrize("n,m,C", [(20, 64, 2), (50, 200, 2), (37, 300, 4), (25, 600, 8)])
def test_emu_fp32_multi_block(default_params, n, m, C):
    rng = np.random.default_rng(n * 1000 + m + 1)
    x = rng.integers(0, 20, size=n).astype(np.uint8)
    y = rng.integers(0, 20, size=m).astype(np.uint8)
    _check(default_params, x, y, C)


def test_emu_related_family_pairs_and_distance_accuracy(default_params):
    fam = inputs.config_family(0)
    for (a, b) in [(0, 1), (2, 5), (6, 7), (1, 4)]:
        _check(default_params, fam.seq(a), fam.seq(b), 4, d_rtol=5e-5)
        r, ref = _check(default_params, fam.seq(a), fam.seq(b), 4, fp64=True, p_tol=1e-7, d_rtol=1e-6)
        assert abs(r.dist - ref.dist) <= 1e-5 * ref.dist   # fp64 mode meets the relative bound even at d ~ 0.01


def test_emu_generic_two_insert_pf_and_fp64(default_params):
    rng = np.random.default_rng(5)
    prm = inputs.Params(hmm=inputs.random_model(rng, 1, 20), pf=inputs.random_model(rng, 2, 20), threshold=0.02)
    x = rng.integers(0, 20, size=45).astype(np.uint8)
    y = rng.integers(0, 20, size=80).astype(np.uint8)
    _check(prm, x, y, 6, GP=2)
    _check(prm, x, y, 2, GP=2)      # multi-block
    _check(prm, x, y, 4, fp64=True, p_tol=1e-7, d_rtol=1e-9)
    _check(prm, x, y, 2, fp64=True, p_tol=1e-7, d_rtol=1e-9)


def test_emu_long_gap_dynamic_range(default_params):
    # 12 vs 400 residues: every path carries ~390 gap residues; plain fp32 would underflow without the exponents
    rng = np.random.default_rng(6)
    x = rng.integers(0, 20, size=12).astype(np.uint8)
    y = rng.integers(0, 20, size=400).astype(np.uint8)
    _check(default_params, x, y, 16)
    _check(default_params, y, x, 2)
    _check(default_params, y, x, 2, mask=1)   # renormalise every 2nd step: same result
