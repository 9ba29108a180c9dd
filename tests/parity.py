"""Shared comparison of the CUDA path's outputs with the oracle (used by the -m gpu tests, smoke() and bench.py)."""
import numpy as np

P_ATOL = 1e-4        # BASELINE.json north_star: dense posteriors max abs error <= 1e-4
D_RTOL = 1e-5        # distances: relative error <= 1e-5
BAND = 1e-4          # sparse pattern identical except entries within 1e-4 of the threshold


def check_pair(ref_dense, ref_dist, ref_logZ, tau, rp, col, val, dist, dense=None, logZ=None, p_atol=P_ATOL,
               d_rtol=D_RTOL, logz_rtol=2e-6, logz_atol=None):
    """Raises AssertionError with a readable message; returns (max |dP|, rel d error)."""
    n, m = ref_dense.shape
    assert len(rp) == n + 1 and rp[0] == 0 and rp[-1] == len(col) == len(val), "row_ptr inconsistent"
    assert (np.diff(rp) >= 0).all(), "row_ptr not monotone"
    rows = np.repeat(np.arange(n), np.diff(rp))
    assert ((col >= 0) & (col < m)).all(), "column out of range"
    for i in np.nonzero(np.diff(rp) > 1)[0]:
        assert (np.diff(col[rp[i]:rp[i + 1]]) > 0).all(), f"columns of row {i} not strictly ascending"
    got = np.zeros((n, m), dtype=bool)
    got[rows, col] = True
    must, may = ref_dense >= tau + BAND, ref_dense >= tau - BAND
    assert got[must].all(), f"{(must & ~got).sum()} entries >= tau+band missing"
    assert not (got & ~may).any(), f"{(got & ~may).sum()} entries < tau-band present"
    err = np.abs(val - ref_dense[rows, col]).max() if len(val) else 0.0
    assert err <= p_atol, f"CSR value error {err:.3e}"
    if dense is not None:
        derr = np.abs(dense - ref_dense).max()
        assert derr <= p_atol, f"dense P error {derr:.3e}"
        err = max(err, derr)
    rel = abs(dist - ref_dist) / max(ref_dist, 1e-300)
    assert rel <= d_rtol or abs(dist - ref_dist) <= 6e-8, f"distance {dist!r} vs {ref_dist!r}: rel {rel:.3e}"
    if logZ is not None:
        # ln Z can be close to 0 (short sequences), so allow an absolute term of the same size as the relative one
        np.testing.assert_allclose(logZ, ref_logZ, rtol=logz_rtol, atol=logz_atol if logz_atol is not None else 10 * logz_rtol)
    return err, rel
