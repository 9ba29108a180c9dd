"""Oracle for stage III, the selective consistency transformation -- TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules
as oracle/qp_oracle.py: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import it; it shares no
code with paper_1512_07437_b200/csrc and neither imports the other).

What it computes, written out plainly in fp64 with scipy.sparse as the matrix-product primitive:

  * PAPER.md:53 (Selective consistency): "consistency relies on the relaxation of posterior probability matrices by
    other sequences" -- S_xy is relaxed over a third sequence z by the product S_xz * S_zy (cost Theta(k^3 n^3) over
    all x, y, z; PAPER.md:59 footnote: sparse matrices).
  * "posterior matrix S_xy is relaxed over sequence z if assumed function f(d_xz, d_yz) fulfills given
    condition"; d = the tree-guided distance ("a number of nodes in a minimal subtree containing both x and y"),
    f = maximum, minimum or sum, thresholded deterministically: relax over z iff f(d_xz, d_yz) <= T
    (Figure 2: accepted "as f(d_xz, d_zy) <= T"; maximum, T ~ 200 is the best setting).
  * PAPER.md:57 / :65: the original signal is amplified "by multiplying S_xy elements by coefficient h_xy. The value
    of h_xy varies from 1 when no relaxations of S_xy are performed, to h when maximum number of relaxations under
    chosen selectivity settings is done (200 in our case)"; h = 3.
  * "the number of transformations is adjusted to the number of sequences (2 for k < 50, 1 otherwise)".

The paper prints no formula for the relaxed matrix. Readings (DESIGN.md section 2b lists them):
  R1  S'_xy = ( 2 h_xy S_xy + sum_{z in sel(x,y)} S_xz S_zy ) / ( 2 h_xy + |sel(x,y)| ).
      With h = 1 and every z selected this is the textbook consistency transformation
      S'_xy = (1/k) sum_{z in all k sequences} S_xz S_zy with S_xx = S_yy = I (the two terms z = x and z = y are each
      S_xy, hence the 2): pinned against exactly that, written as ONE block-matrix product, in
      tests/test_consistency_oracle_pins.py. "Multiplying S_xy elements by h_xy" scales those two terms; dividing by
      the total weight keeps S' an average (entries stay in [0, 1] whatever |sel| is), which is what "sets of
      different sizes [are] handled properly" asks for.
  R2  h_xy = 1 + (h - 1) * min(r, R) / R, r = |sel(x,y)|, R = 200: linear between the two end points the paper gives.
  R3  S_zx = S_xz^T for the pair stored the other way round; pairs that are not in the input are never relaxed over
      (z is selected only if both (x,z) and (z,y) are present).
  R4  The relaxed matrix keeps the sparsity pattern of S_xy (only cells that are non-zero in S_xy are computed: this
      is what bounds the cost by the footnote's beta factors) and drops relaxed values below the stage-I threshold tau.
  R5  All matrices of one transformation are computed from the matrices BEFORE it (Jacobi style); the second
      transformation of small sets (k < 50) repeats the same step on the result.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

SEL_MAX, SEL_MIN, SEL_SUM = 0, 1, 2


def oriented(S, a, b):
    """S_ab as a CSR matrix with rows = residues of a (R3): stored as (a, b), or the transpose of the stored (b, a)."""
    if (a, b) in S:
        return S[(a, b)]
    return S[(b, a)].T.tocsr()


def present(S, a, b):
    return (a, b) in S or (b, a) in S


def f_value(dxz, dyz, f):
    """'Maximum, minimum, or sum can be used as examples of f function'."""
    if f == SEL_MAX:
        return max(dxz, dyz)
    if f == SEL_MIN:
        return min(dxz, dyz)
    return dxz + dyz


def select(S, k, treedist, x, y, T, f=SEL_MAX):
    """sel(x, y): the sequences z (ascending) S_xy is relaxed over: f(d_xz, d_yz) <= T and both pairs present."""
    return [z for z in range(k) if z != x and z != y and present(S, x, z) and present(S, z, y)
            and f_value(int(treedist[x, z]), int(treedist[y, z]), f) <= T]


def h_coefficient(r, h=3.0, max_relax=200):
    """R2: 1 when nothing is relaxed, h at max_relax relaxations or more, linear in between."""
    return 1.0 + (h - 1.0) * min(r, max_relax) / float(max_relax)


def relax_pair(S, x, y, zs, h_xy, tau):
    """R1 + R4 for one stored pair (x, y): returns the relaxed CSR matrix (fp64)."""
    Sxy = S[(x, y)].tocsr()
    acc = (2.0 * h_xy) * Sxy
    for z in zs:
        acc = acc + oriented(S, x, z) @ oriented(S, z, y)      # S_xz S_zy: a library sparse product
    acc = acc / (2.0 * h_xy + len(zs))
    pattern = Sxy.copy()
    pattern.data[:] = 1.0
    out = sp.csr_matrix(acc).multiply(pattern).tocsr()         # R4: only the cells of S_xy's pattern
    out.data[out.data < tau] = 0.0                             # ... and of those, the values >= tau
    out.eliminate_zeros()
    out.sort_indices()
    return out


def transform(S, k, treedist, T=200, f=SEL_MAX, h=3.0, max_relax=200, tau=0.01):
    """One consistency transformation (R5) of every stored pair. S: {(x, y): csr}. Returns (S', relaxations[(x, y)])."""
    out, count = {}, {}
    for (x, y) in S:
        zs = select(S, k, treedist, x, y, T, f)
        out[(x, y)] = relax_pair(S, x, y, zs, h_coefficient(len(zs), h, max_relax), tau)
        count[(x, y)] = len(zs)
    return out, count


def n_transformations(k):
    """2 for k < 50, 1 otherwise."""
    return 2 if k < 50 else 1


def from_csr(rp, col, val, n, m):
    """A stage-I pair (row_ptr, col, val) as scipy CSR, fp64."""
    return sp.csr_matrix((np.asarray(val, dtype=np.float64), np.asarray(col, dtype=np.int32),
                          np.asarray(rp, dtype=np.int32)), shape=(int(n), int(m)))
