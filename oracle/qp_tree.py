"""Oracle for stage II -- TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/qp_oracle.py: only tests/,
__graft_entry__.smoke() and bench.py's CPU legs may import it; it shares no code with paper_1512_07437_b200/csrc).

What it computes, written out plainly:
  * PAPER.md:23 (Methods): "pairwise distances ... are given as an input for weighted UPGMA algorithm [ref 19, :225]
    for guide tree construction". Weighted UPGMA (WPGMA): start with k singleton clusters; repeatedly merge the two
    closest clusters i, j into a new one u with d(u, m) = (d(i, m) + d(j, m)) / 2 for every other cluster m; the
    height of u is d(i, j). k - 1 merges.
  * PAPER.md:55 (selective consistency): the tree-guided distance of x and y is "a number of nodes in a minimal
    subtree containing both x and y", i.e. the node count of the subtree rooted at their lowest common ancestor
    (Figure 2: "At each node, a size of a subtree is given").

Readings: (1) "number of nodes" counts leaves AND internal nodes: 2 * leaves - 1;
(2) ties between equal distances are broken towards the lexicographically smallest cluster pair (i < j, cluster
numbers as below) -- the paper is silent, any rule gives a valid weighted-UPGMA tree; (3) the averages are taken in
IEEE fp32, the precision the distances arrive in from stage I: an argmin over floating-point values is a decision,
so both sides take it in the same precision (the kernel's).

Node numbering: leaves 0..k-1, the node created by merge t (t = 0..k-2) is k + t. A cluster keeps the SLOT of its
smaller-numbered child (slot = the index of one of its leaves in the working matrix), so "cluster pair (i, j)" above
means slots i < j.
"""
from __future__ import annotations

import numpy as np


def wpgma(dist):
    """dist: k x k symmetric, only the off-diagonal entries are read. Returns
    merge int32[k-1][2] (node ids of the children, the one in the smaller slot first), height float32[k-1],
    leaves int32[2k-1] (leaf count of every node), parent int32[2k-1] (-1 for the root)."""
    D = np.array(dist, dtype=np.float32, copy=True)
    k = D.shape[0]
    node = np.arange(k)              # node id currently living in slot s
    alive = np.ones(k, dtype=bool)
    merge = np.zeros((max(k - 1, 0), 2), dtype=np.int32)
    height = np.zeros(max(k - 1, 0), dtype=np.float32)
    leaves = np.ones(2 * k - 1, dtype=np.int32)
    parent = -np.ones(2 * k - 1, dtype=np.int32)
    upper = np.triu(np.ones((k, k), dtype=bool), 1)
    for t in range(k - 1):
        # the closest pair of live clusters; np.argmin returns the FIRST minimum of the row-major scan, i.e. the
        # lexicographically smallest (i, j), i < j, among equal distances
        M = np.where(upper & alive[:, None] & alive[None, :], D, np.float32(np.inf))
        i, j = divmod(int(np.argmin(M)), k)
        u = k + t
        merge[t] = (node[i], node[j])
        height[t] = D[i, j]
        leaves[u] = leaves[node[i]] + leaves[node[j]]
        parent[node[i]] = parent[node[j]] = u
        v = ((D[i, :] + D[j, :]) * np.float32(0.5)).astype(np.float32)   # fp32 add, fp32 multiply by 1/2 (exact)
        others = alive.copy()
        others[i] = others[j] = False
        D[i, others] = v[others]
        D[others, i] = v[others]
        alive[j] = False
        node[i] = u
    return merge, height, leaves, parent


def tree_distance(leaves, parent, k):
    """int32 k x k: node count (2 * leaves - 1) of the subtree rooted at the lowest common ancestor; diagonal 1."""
    anc = []
    for x in range(k):
        a, chain = x, []
        while a != -1:
            chain.append(a)
            a = int(parent[a])
        anc.append(chain)
    T = np.ones((k, k), dtype=np.int32)
    for x in range(k):
        sx = set(anc[x])
        for y in range(k):
            if x != y:
                lca = next(a for a in anc[y] if a in sx)
                T[x, y] = 2 * int(leaves[lca]) - 1
    return T
