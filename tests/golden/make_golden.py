"""Writes tests/golden/cfg0_oracle.txt: regression values of the ORACLE on BASELINE.json configs[0]
(8 synthetic proteins, all 28 pairs, default model, tau = 0.01).

    python tests/golden/make_golden.py

Calls only oracle/ (plus the seeded input generator); nothing here comes from the CUDA path. The paper
(stage I) prints no worked numeric example, so these are not paper values: they pin the oracle
against accidental change (a later edit of its arithmetic must regenerate this file and say why in the commit).
Columns: x y n m nnz distance lnZ_hmm lnZ_pf sum(P) max(P)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import qp_oracle as orc  # noqa: E402
from paper_1512_07437_b200 import inputs  # noqa: E402


def rows():
    prm = inputs.default_params()
    fam = inputs.config_family(0)
    pairs = inputs.all_pairs(fam.k)
    run = orc.Run(prm, fam, pairs, keep_dense=True)
    L = fam.lengths
    for p, (a, b) in enumerate(pairs):
        P = run.dense(p)
        z = run.logZ(p)
        yield (int(a), int(b), int(L[a]), int(L[b]), int(run.nnz[p]), float(run.dist[p]), float(z[0]), float(z[2]),
               float(P.sum()), float(P.max()))


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle.txt")
    with open(out, "w") as f:
        f.write("# oracle regression values, BASELINE.json configs[0] (seed 7437000), default model, tau 0.01\n")
        f.write("# written by tests/golden/make_golden.py from oracle/ only; not paper values (PAPER.md prints none)\n")
        f.write("# x y n m nnz distance lnZ_hmm lnZ_pf sumP maxP\n")
        for r in rows():
            f.write("%d %d %d %d %d %.15e %.15e %.15e %.15e %.15e\n" % r)
    print(out)


if __name__ == "__main__":
    main()
