"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NO arithmetic of the method (no recurrence, no posterior, no distance). It only makes
inputs: residue strings of synthetic protein families (SURVEY.md §8(d) recipe, standing in for the paper's
BAliBASE/PREFAB/OXBench/SABmark/BaliFam/HomFam families, which are not available) and the
parameter values of the two probabilistic models (the paper names its tables but never
prints them, so they are inputs here).

Every function is deterministic in its seed (numpy PCG64).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

ALPHABET = 20
SEED_BASE = 7437000  # seed = SEED_BASE + config index

NEG_INF = float("-inf")


# --------------------------------------------------------------------------------------------------------------
# model parameter values (inputs; SURVEY.md §8(c) c-1 for the meaning of each field, c-5 for the default values)
# --------------------------------------------------------------------------------------------------------------
@dataclass
class Model:
    """One weighted pair automaton in natural-log weights (field meaning: include/qp.h `qp_model`)."""

    n_ins: int
    alphabet: int
    log_match: np.ndarray  # [A, A] float64, symmetric
    log_ins: np.ndarray  # [A] float64
    t_MM: float
    t_MI: tuple
    t_II: tuple
    t_IM: tuple
    init_M: float
    init_I: tuple
    end_M: float
    end_I: tuple

    def padded(self, name: str):
        """Length-2 list of a per-insert-state field; unused slots are -inf (weight 0)."""
        v = list(getattr(self, name))
        return v + [NEG_INF] * (2 - len(v))


@dataclass
class Params:
    hmm: Model
    pf: Model
    threshold: float = 0.01


def background(alphabet: int = ALPHABET) -> np.ndarray:
    """q_a ∝ 2 + ((7a+3) mod 11)  (c-5)."""
    w = np.array([2 + ((7 * a + 3) % 11) for a in range(alphabet)], dtype=np.float64)
    return w / w.sum()


def joint_emission(q: np.ndarray, lam: float) -> np.ndarray:
    """F81-type joint table e(a,b) = q_a (lam [a=b] + (1-lam) q_b): symmetric, sums to 1 (c-5)."""
    return q[:, None] * (lam * np.eye(len(q)) + (1.0 - lam) * q[None, :])


def default_hmm(alphabet: int = ALPHABET, lam: float = 0.40, delta=(0.020, 0.005), eps=(0.60, 0.95),
                pi=(0.15, 0.05)) -> Model:
    """Pair-HMM instance, G = len(delta) insert-state pairs (c-1 'HMM instance', c-5 values)."""
    q = background(alphabet)
    e = joint_emission(q, lam)
    g = len(delta)
    return Model(
        n_ins=g, alphabet=alphabet, log_match=np.log(e), log_ins=np.log(q),
        t_MM=math.log(1.0 - 2.0 * sum(delta)),
        t_MI=tuple(math.log(d) for d in delta),
        t_II=tuple(math.log(x) for x in eps),
        t_IM=tuple(math.log(1.0 - x) for x in eps),
        init_M=math.log(1.0 - 2.0 * sum(pi)), init_I=tuple(math.log(p) for p in pi),
        end_M=math.log(1.0 - 2.0 * sum(pi)), end_I=tuple(math.log(p) for p in pi),
    )


def default_pf(alphabet: int = ALPHABET, lam: float = 0.25, gap_open: float = 11.0, gap_ext: float = 1.0,
               temperature: float = 3.0) -> Model:
    """Partition-function instance, already divided by the temperature (c-1 'PF instance', c-5 values)."""
    q = background(alphabet)
    e = joint_emission(q, lam)
    s = (2.0 / math.log(2.0)) * np.log(e / (q[:, None] * q[None, :]))  # half-bit log-odds, unrounded
    return Model(
        n_ins=1, alphabet=alphabet, log_match=s / temperature, log_ins=np.zeros(alphabet),
        t_MM=0.0, t_MI=(-gap_open / temperature,), t_II=(-gap_ext / temperature,), t_IM=(0.0,),
        init_M=0.0, init_I=(-gap_open / temperature,), end_M=0.0, end_I=(0.0,),
    )


def default_params(threshold: float = 0.01) -> Params:
    return Params(hmm=default_hmm(), pf=default_pf(), threshold=threshold)


def nucleotide_params(threshold: float = 0.01) -> Params:
    """Nucleotide mode ("HOXD substitution matrices and GTR evolutionary model"): the same two
    automata over a 4-letter alphabet. The HOXD and GTR tables are not in the container and are not reconstructed;
    this is the synthetic F81-type model of c-5 with A = 4, a stand-in with the right shape."""
    return Params(hmm=default_hmm(alphabet=4, lam=0.55), pf=default_pf(alphabet=4, lam=0.45, gap_open=8.0),
                  threshold=threshold)


def random_model(rng: np.random.Generator, n_ins: int, alphabet: int = 4) -> Model:
    """A random symmetric model for parameter-agnostic pins (brute force, fwd=bwd, transposition)."""
    lm = rng.normal(0.0, 1.0, size=(alphabet, alphabet))
    lm = 0.5 * (lm + lm.T)
    return Model(
        n_ins=n_ins, alphabet=alphabet, log_match=lm, log_ins=rng.normal(-1.0, 0.5, size=alphabet),
        t_MM=float(rng.normal(-0.2, 0.3)),
        t_MI=tuple(float(v) for v in rng.normal(-2.0, 0.7, size=n_ins)),
        t_II=tuple(float(v) for v in rng.normal(-0.7, 0.4, size=n_ins)),
        t_IM=tuple(float(v) for v in rng.normal(-0.5, 0.4, size=n_ins)),
        init_M=float(rng.normal(-0.5, 0.3)), init_I=tuple(float(v) for v in rng.normal(-2.0, 0.5, size=n_ins)),
        end_M=float(rng.normal(-0.5, 0.3)), end_I=tuple(float(v) for v in rng.normal(-2.0, 0.5, size=n_ins)),
    )


# --------------------------------------------------------------------------------------------------------------
# synthetic protein families (SURVEY.md §8(d) `gen_family`)
# --------------------------------------------------------------------------------------------------------------
@dataclass
class Family:
    """Packed residue codes: sequence s is seqs[offsets[s]:offsets[s+1]]."""

    seqs: np.ndarray  # uint8 [total]
    offsets: np.ndarray  # int64 [k+1]
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def k(self) -> int:
        return len(self.offsets) - 1

    @property
    def lengths(self) -> np.ndarray:
        return np.diff(self.offsets)

    def seq(self, s: int) -> np.ndarray:
        return self.seqs[self.offsets[s]:self.offsets[s + 1]]


def pack(seq_list) -> Family:
    offs = np.zeros(len(seq_list) + 1, dtype=np.int64)
    for i, s in enumerate(seq_list):
        offs[i + 1] = offs[i] + len(s)
    flat = np.concatenate([np.asarray(s, dtype=np.uint8) for s in seq_list]) if seq_list else np.zeros(0, np.uint8)
    return Family(seqs=np.ascontiguousarray(flat, dtype=np.uint8), offsets=offs)


def _coalescent(k: int, rng: np.random.Generator, deep: bool):
    """Ultrametric tree, root height 1: Kingman topology, heights sorted U(0,1) ('deep': U^(1/3)), top = 1."""
    if k == 1:
        return [(-1, -1)], np.zeros(1), 0
    h = rng.random(k - 1)
    if deep:
        h = h ** (1.0 / 3.0)
    h = np.sort(h)
    h[-1] = 1.0
    children = [(-1, -1)] * k
    height = [0.0] * k
    live = list(range(k))
    for step in range(k - 1):
        a, b = rng.choice(len(live), size=2, replace=False)
        na, nb = live[a], live[b]
        for idx in sorted((a, b), reverse=True):
            live.pop(idx)
        children.append((na, nb))
        height.append(float(h[step]))
        live.append(len(children) - 1)
    return children, np.asarray(height), live[0]


def _evolve(seq: np.ndarray, t: float, q, r_sub, r_indel, indel_mean, rng) -> np.ndarray:
    seq = seq.copy()
    if t <= 0.0:
        return seq
    p_sub = 1.0 - (1.0 - r_sub) ** t
    hit = rng.random(len(seq)) < p_sub
    nh = int(hit.sum())
    if nh:
        seq[hit] = rng.choice(len(q), size=nh, p=q).astype(np.uint8)
    n_ev = int(rng.poisson(r_indel * t * len(seq)))
    for _ in range(n_ev):
        ln = int(rng.geometric(1.0 / indel_mean))
        if rng.random() < 0.5:  # insertion
            pos = int(rng.integers(0, len(seq) + 1))
            ins = rng.choice(len(q), size=ln, p=q).astype(np.uint8)
            seq = np.concatenate([seq[:pos], ins, seq[pos:]])
        elif len(seq) > ln + 1:  # deletion (never delete everything)
            pos = int(rng.integers(0, len(seq) - ln + 1))
            seq = np.concatenate([seq[:pos], seq[pos + ln:]])
    return seq


def gen_family(k: int, length_law, r_sub: float, r_indel: float, seed: int, indel_mean: float = 3.0,
               tree: str = "random", name: str = "") -> Family:
    """SURVEY.md §8(d) steps 1-5. `length_law(rng, k)` returns k real target lengths."""
    rng = np.random.Generator(np.random.PCG64(seed))
    q = background()
    L = np.maximum(np.rint(length_law(rng, k)).astype(np.int64), 20)
    root = rng.choice(ALPHABET, size=int(L.max()), p=q).astype(np.uint8)
    children, height, root_id = _coalescent(k, rng, deep=(tree == "deep"))
    node_seq = {root_id: root}
    stack = [root_id]
    leaves = [None] * k
    while stack:
        nd = stack.pop()
        s = node_seq.pop(nd)
        if nd < k:
            leaves[nd] = s
            continue
        for ch in children[nd]:
            node_seq[ch] = _evolve(s, float(height[nd] - height[ch]), q, r_sub, r_indel, indel_mean, rng)
            stack.append(ch)
    out = []
    for i in range(k):
        s = leaves[i]
        w = int(min(L[i], len(s)))
        mid = len(s) // 2 + int(rng.integers(-(L[i] // 4), L[i] // 4 + 1))
        start = min(max(mid - w // 2, 0), len(s) - w)
        out.append(s[start:start + w])
    fam = pack(out)
    fam.name = name
    fam.meta = dict(k=k, r_sub=r_sub, r_indel=r_indel, indel_mean=indel_mean, tree=tree, seed=seed)
    return fam


_CONFIGS = {
    # BASELINE.json configs[0..4]; concrete laws from SURVEY.md §8(d)
    0: dict(k=8, law=lambda r, k: r.integers(60, 101, size=k).astype(float), r_sub=0.3, r_indel=0.05, tree="random"),
    1: dict(k=50, law=lambda r, k: r.normal(250.0, 50.0, size=k), r_sub=0.5, r_indel=0.05, tree="random"),
    2: dict(k=200, law=lambda r, k: r.normal(300.0, 60.0, size=k), r_sub=0.6, r_indel=0.08, tree="random"),
    3: dict(k=1000, law=lambda r, k: r.normal(350.0, 80.0, size=k), r_sub=0.7, r_indel=0.05, tree="deep"),
    4: dict(k=120, law=lambda r, k: np.exp(r.uniform(math.log(50.0), math.log(2000.0), size=k)), r_sub=0.5,
            r_indel=0.05, tree="random"),
}


def config_family(cfg: int) -> Family:
    """The seeded synthetic family of BASELINE.json configs[cfg] (seed 7437000 + cfg)."""
    c = _CONFIGS[cfg]
    return gen_family(c["k"], c["law"], c["r_sub"], c["r_indel"], seed=SEED_BASE + cfg, tree=c["tree"],
                      name=f"cfg{cfg}")


def all_pairs(k: int) -> np.ndarray:
    """All x<y pairs, row-major, int32 [k(k-1)/2, 2]."""
    iu = np.triu_indices(k, 1)
    return np.ascontiguousarray(np.stack(iu, axis=1).astype(np.int32))


def random_family(rng: np.random.Generator, k: int, lo: int, hi: int, alphabet: int = ALPHABET) -> Family:
    """k unrelated iid sequences with lengths uniform in [lo, hi] (edge-case and API tests)."""
    return pack([rng.integers(0, alphabet, size=int(rng.integers(lo, hi + 1))).astype(np.uint8) for _ in range(k)])
