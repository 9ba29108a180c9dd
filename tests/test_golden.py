"""The oracle reproduces its stored regression values for configs[0] (tests/golden/cfg0_oracle.txt, written by
tests/golden/make_golden.py from oracle/ only). Guards the oracle and the seeded input generator against silent change."""
import os

import numpy as np

from tests.golden import make_golden

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_matches_golden_cfg0():
    want = np.loadtxt(os.path.join(HERE, "golden", "cfg0_oracle.txt"))
    got = np.array(list(make_golden.rows()))
    assert want.shape == got.shape == (28, 10)
    assert (want[:, :5] == got[:, :5]).all()                      # indices, lengths, nnz: exact
    np.testing.assert_allclose(got[:, 5:], want[:, 5:], rtol=1e-12, atol=0)
