"""Brute-force enumeration of every alignment path of a weighted pair automaton.

Pure Python, linear (non-log) fp64 weights, no dynamic programming: it checks the oracle's recurrences
(oracle/qp_oracle.c) and is itself independent of them. Usable for n, m <= ~6.

A path is a sequence of states s_1..s_L, each M (consumes x_i and y_j), X_g (consumes x_i) or Y_g (consumes
y_j), consuming all of x and y. Allowed moves: M->M, M->X_g, M->Y_g, X_g->X_g, X_g->M, Y_g->Y_g, Y_g->M
(no X<->Y, no X_g->X_g'). weight = init(s_1) * prod emissions * prod transitions * end(s_L).
"""
import math


def _w(v):
    return 0.0 if v == float("-inf") else math.exp(v)


def enumerate_paths(model, x, y):
    """Yield (weight, [(i,j) 1-based match cells]) for every path."""
    n, m, G = len(x), len(y), model.n_ins
    lm, li = model.log_match, model.log_ins
    t_MI, t_II, t_IM = model.padded("t_MI"), model.padded("t_II"), model.padded("t_IM")
    init_I, end_I = model.padded("init_I"), model.padded("end_I")
    out = []

    def trans(prev, cur):
        if prev is None:
            return _w(model.init_M) if cur == ("M",) else _w(init_I[cur[1]])
        if prev == ("M",):
            return _w(model.t_MM) if cur == ("M",) else _w(t_MI[cur[1]])
        if cur == ("M",):
            return _w(t_IM[prev[1]])
        return _w(t_II[cur[1]]) if prev == cur else 0.0

    def rec(i, j, prev, w, cells):
        if i == n and j == m:
            end = _w(model.end_M) if prev == ("M",) else _w(end_I[prev[1]])
            out.append((w * end, list(cells)))
            return
        if i < n and j < m:
            t = trans(prev, ("M",))
            if t > 0.0:
                cells.append((i + 1, j + 1))
                rec(i + 1, j + 1, ("M",), w * t * math.exp(lm[x[i]][y[j]]), cells)
                cells.pop()
        for g in range(G):
            if i < n:
                t = trans(prev, ("X", g))
                if t > 0.0:
                    rec(i + 1, j, ("X", g), w * t * math.exp(li[x[i]]), cells)
            if j < m:
                t = trans(prev, ("Y", g))
                if t > 0.0:
                    rec(i, j + 1, ("Y", g), w * t * math.exp(li[y[j]]), cells)

    rec(0, 0, None, 1.0, [])
    return out


def posterior(model, x, y):
    """(P[n][m] list of lists, Z) by summing path weights."""
    n, m = len(x), len(y)
    paths = enumerate_paths(model, x, y)
    Z = math.fsum(w for w, _ in paths)
    acc = [[[] for _ in range(m)] for _ in range(n)]
    for w, cells in paths:
        for (i, j) in cells:
            acc[i - 1][j - 1].append(w)
    P = [[math.fsum(acc[i][j]) / Z for j in range(m)] for i in range(n)]
    return P, Z


def mea(P):
    """max over all monotone (strictly increasing in both indices) match sets of sum P, by enumeration."""
    n, m = len(P), len(P[0])
    best = [0.0]

    def rec(i, j0, s):
        # rows i.. remain, columns j0.. remain
        if s > best[0]:
            best[0] = s
        if i >= n or j0 >= m:
            return
        rec(i + 1, j0, s)  # row i unmatched
        for j in range(j0, m):
            rec(i + 1, j + 1, s + P[i][j])

    rec(0, 0, 0.0)
    return best[0]
