"""ctypes wrapper over oracle/qp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares no code with paper_1512_07437_b200/csrc or the qp binding; the only thing both sides consume is the
input dataclasses of paper_1512_07437_b200.inputs (sequences and model parameter values).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qp_oracle.c")
_LIB = os.path.join(_HERE, "libqp_oracle.so")


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the oracle into oracle/libqp_oracle.so (no -ffast-math: plain IEEE fp64)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Model(C.Structure):
    _fields_ = [
        ("n_ins", C.c_int32), ("alphabet", C.c_int32),
        ("log_match", C.POINTER(C.c_double)), ("log_ins", C.POINTER(C.c_double)),
        ("t_MM", C.c_double), ("t_MI", C.c_double * 2), ("t_II", C.c_double * 2), ("t_IM", C.c_double * 2),
        ("init_M", C.c_double), ("init_I", C.c_double * 2), ("end_M", C.c_double), ("end_I", C.c_double * 2),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, u8p, i32p, i64p = C.POINTER(C.c_double), C.POINTER(C.c_uint8), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        mp = C.POINTER(_Model)
        L.qpo_forward.restype = C.c_double
        L.qpo_forward.argtypes = [mp, u8p, C.c_int, u8p, C.c_int, dp]
        L.qpo_backward.restype = C.c_double
        L.qpo_backward.argtypes = [mp, u8p, C.c_int, u8p, C.c_int, dp]
        L.qpo_posterior.restype = None
        L.qpo_posterior.argtypes = [mp, u8p, C.c_int, u8p, C.c_int, dp, dp, dp, dp, dp]
        L.qpo_combine.restype = None
        L.qpo_combine.argtypes = [dp, dp, C.c_size_t, dp]
        L.qpo_mea.restype = C.c_double
        L.qpo_mea.argtypes = [dp, C.c_int, C.c_int]
        L.qpo_distance.restype = C.c_double
        L.qpo_distance.argtypes = [C.c_double, C.c_int, C.c_int]
        L.qpo_pair.restype = C.c_double
        L.qpo_pair.argtypes = [mp, mp, u8p, C.c_int, u8p, C.c_int, dp, dp, dp, dp]
        L.qpo_run.restype = C.c_void_p
        L.qpo_run.argtypes = [mp, mp, C.c_double, u8p, i64p, i32p, C.c_int64, C.c_int, C.c_int]
        L.qpo_result_nnz.restype = C.c_int64
        L.qpo_result_nnz.argtypes = [C.c_void_p, C.c_int64]
        L.qpo_result_rows.restype = C.c_int32
        L.qpo_result_rows.argtypes = [C.c_void_p, C.c_int64]
        L.qpo_result_threads.restype = C.c_int
        L.qpo_result_threads.argtypes = [C.c_void_p]
        L.qpo_result_seconds.restype = C.c_double
        L.qpo_result_seconds.argtypes = [C.c_void_p]
        L.qpo_result_dist.restype = C.c_double
        L.qpo_result_dist.argtypes = [C.c_void_p, C.c_int64]
        L.qpo_result_logZ.restype = None
        L.qpo_result_logZ.argtypes = [C.c_void_p, C.c_int64, dp]
        L.qpo_result_csr.restype = None
        L.qpo_result_csr.argtypes = [C.c_void_p, C.c_int64, i32p, i32p, dp]
        L.qpo_result_dense.restype = C.c_int
        L.qpo_result_dense.argtypes = [C.c_void_p, C.c_int64, dp, C.c_int64]
        L.qpo_result_free.restype = None
        L.qpo_result_free.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _u8(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint8))


class CModel:
    """Keeps the numpy buffers alive next to the C struct."""

    def __init__(self, m):
        self.lm = np.ascontiguousarray(m.log_match, dtype=np.float64)
        self.li = np.ascontiguousarray(m.log_ins, dtype=np.float64)
        s = _Model()
        s.n_ins, s.alphabet = int(m.n_ins), int(m.alphabet)
        s.log_match, s.log_ins = _dp(self.lm), _dp(self.li)
        s.t_MM, s.init_M, s.end_M = float(m.t_MM), float(m.init_M), float(m.end_M)
        for name in ("t_MI", "t_II", "t_IM", "init_I", "end_I"):
            arr = getattr(s, name)
            for g, v in enumerate(m.padded(name)):
                arr[g] = v
        self.s = s
        self.n_states = 1 + 2 * s.n_ins

    @property
    def ref(self):
        return C.byref(self.s)


def _seq(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


def forward(model, x, y):
    """All forward planes [S, n+1, m+1] (state order M, X_1..X_G, Y_1..Y_G) and logZ_f."""
    cm, x, y = CModel(model), _seq(x), _seq(y)
    F = np.empty((cm.n_states, len(x) + 1, len(y) + 1))
    z = lib().qpo_forward(cm.ref, _u8(x), len(x), _u8(y), len(y), _dp(F))
    return F, z


def backward(model, x, y):
    cm, x, y = CModel(model), _seq(x), _seq(y)
    B = np.empty((cm.n_states, len(x) + 1, len(y) + 1))
    z = lib().qpo_backward(cm.ref, _u8(x), len(x), _u8(y), len(y), _dp(B))
    return B, z


def posterior(model, x, y):
    """Dense P_model [n, m], logZ_f, logZ_b, and the planes F, B."""
    cm, x, y = CModel(model), _seq(x), _seq(y)
    n, m = len(x), len(y)
    F = np.empty((5, n + 1, m + 1))
    B = np.empty((5, n + 1, m + 1))
    P = np.empty((n, m))
    zf, zb = C.c_double(), C.c_double()
    lib().qpo_posterior(cm.ref, _u8(x), n, _u8(y), m, _dp(F), _dp(B), _dp(P), C.byref(zf), C.byref(zb))
    S = cm.n_states
    Fv = F.reshape(-1)[: S * (n + 1) * (m + 1)].reshape(S, n + 1, m + 1)
    Bv = B.reshape(-1)[: S * (n + 1) * (m + 1)].reshape(S, n + 1, m + 1)
    return P, zf.value, zb.value, Fv, Bv


def combine(Ph, Pp):
    Ph, Pp = np.ascontiguousarray(Ph, dtype=np.float64), np.ascontiguousarray(Pp, dtype=np.float64)
    out = np.empty_like(Ph)
    lib().qpo_combine(_dp(Ph), _dp(Pp), Ph.size, _dp(out))
    return out


def mea(P):
    P = np.ascontiguousarray(P, dtype=np.float64)
    return lib().qpo_mea(_dp(P), P.shape[0], P.shape[1])


def distance(mea_score, n, m):
    return lib().qpo_distance(float(mea_score), int(n), int(m))


@dataclass
class PairResult:
    P: np.ndarray
    Ph: np.ndarray
    Pp: np.ndarray
    logZ: np.ndarray  # hmm fwd, hmm bwd, pf fwd, pf bwd
    dist: float


def pair(params, x, y) -> PairResult:
    h, p, x, y = CModel(params.hmm), CModel(params.pf), _seq(x), _seq(y)
    n, m = len(x), len(y)
    P, Ph, Pp, z = np.empty((n, m)), np.empty((n, m)), np.empty((n, m)), np.empty(4)
    d = lib().qpo_pair(h.ref, p.ref, _u8(x), n, _u8(y), m, _dp(P), _dp(Ph), _dp(Pp), _dp(z))
    return PairResult(P=P, Ph=Ph, Pp=Pp, logZ=z, dist=d)


class Run:
    """All listed pairs: per-pair CSR (P >= tau), distances, logZ; optional dense P. Frees the C handle on del."""

    def __init__(self, params, family, pairs, keep_dense=False, threads=0):
        self._h = None
        h, p = CModel(params.hmm), CModel(params.pf)
        self.pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        self.family = family
        seqs = np.ascontiguousarray(family.seqs, dtype=np.uint8)
        offs = np.ascontiguousarray(family.offsets, dtype=np.int64)
        self._h = lib().qpo_run(h.ref, p.ref, float(params.threshold), _u8(seqs),
                                offs.ctypes.data_as(C.POINTER(C.c_int64)),
                                self.pairs.ctypes.data_as(C.POINTER(C.c_int32)), len(self.pairs),
                                int(bool(keep_dense)), int(threads))
        self.n_pairs = len(self.pairs)
        self.threads = lib().qpo_result_threads(self._h)
        self.seconds = lib().qpo_result_seconds(self._h)
        self.dist = np.array([lib().qpo_result_dist(self._h, i) for i in range(self.n_pairs)])
        self.nnz = np.array([lib().qpo_result_nnz(self._h, i) for i in range(self.n_pairs)], dtype=np.int64)
        self.rows = np.array([lib().qpo_result_rows(self._h, i) for i in range(self.n_pairs)], dtype=np.int64)

    def logZ(self, p):
        z = np.empty(4)
        lib().qpo_result_logZ(self._h, p, _dp(z))
        return z

    def csr(self, p):
        rp = np.empty(self.rows[p] + 1, dtype=np.int32)
        col = np.empty(self.nnz[p], dtype=np.int32)
        val = np.empty(self.nnz[p], dtype=np.float64)
        lib().qpo_result_csr(self._h, p, rp.ctypes.data_as(C.POINTER(C.c_int32)),
                             col.ctypes.data_as(C.POINTER(C.c_int32)), _dp(val))
        return rp, col, val

    def dense(self, p):
        L = self.family.lengths
        n, m = int(L[self.pairs[p, 0]]), int(L[self.pairs[p, 1]])
        out = np.empty((n, m))
        if lib().qpo_result_dense(self._h, p, _dp(out), n * m) != 0:
            raise RuntimeError("dense P was not kept (keep_dense=False)")
        return out

    def dist_matrix(self):
        k = self.family.k
        D = np.zeros((k, k))
        D[self.pairs[:, 0], self.pairs[:, 1]] = self.dist
        D[self.pairs[:, 1], self.pairs[:, 0]] = self.dist
        return D

    def __del__(self):
        if getattr(self, "_h", None):
            try:
                lib().qpo_result_free(self._h)
            except TypeError:   # interpreter shutdown: the module globals are already gone, the process frees the memory
                pass
            self._h = None
