"""ctypes driver for tests/simt_emu/emu.cpp (CPU lockstep emulation of the CUDA lane code; test harness only)."""
import ctypes as C
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(os.path.dirname(_HERE))
_SRC = os.path.join(_HERE, "emu.cpp")
_LIB = os.path.join(_HERE, "libemu.so")
_HDR = os.path.join(_ROOT, "paper_1512_07437_b200", "csrc", "qp_lane.h")


def build():
    if not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)):
        subprocess.run(["g++", "-O2", "-std=c++17", "-mfma", "-ffp-contract=off", "-fPIC", "-shared",
                        "-I" + os.path.dirname(_HDR), "-o", _LIB, _SRC], check=True)
    return _LIB


class EmuModel(C.Structure):
    _fields_ = [("em", C.c_double * 1024), ("wMM", C.c_double), ("wMI", C.c_double * 2), ("wII", C.c_double * 2),
                ("wIM", C.c_double * 2), ("initM", C.c_double), ("initI", C.c_double * 2), ("endM", C.c_double),
                ("endI", C.c_double * 2)]


def _ex(v):
    return 0.0 if v == float("-inf") else math.exp(v)


def make_model(m):
    """Linear weights + background-normalised emission table (the same preparation qp_api.cu does on the host)."""
    s = EmuModel()
    A = m.alphabet
    lo = m.log_match - m.log_ins[:, None] - m.log_ins[None, :]
    for a in range(A):
        for b in range(A):
            s.em[a * 32 + b] = _ex(lo[a, b])
    s.wMM, s.initM, s.endM = _ex(m.t_MM), _ex(m.init_M), _ex(m.end_M)
    for name, f in (("t_MI", "wMI"), ("t_II", "wII"), ("t_IM", "wIM"), ("init_I", "initI"), ("end_I", "endI")):
        for g, v in enumerate(m.padded(name)):
            getattr(s, f)[g] = _ex(v)
    return s


class EmuResult:
    pass


def run(params, x, y, C_, fp64=False, GP=None, mask=7):
    L = C.CDLL(build())
    L.emu_run.restype = C.c_int
    x = np.ascontiguousarray(x, dtype=np.uint8)
    y = np.ascontiguousarray(y, dtype=np.uint8)
    n, m = len(x), len(y)
    mh, mp = make_model(params.hmm), make_model(params.pf)
    GP = GP if GP is not None else (2 if fp64 else params.pf.n_ins)
    dense = np.zeros((n, m), dtype=np.float32)
    lz, dist = (C.c_double * 4)(), C.c_double()
    rc = L.emu_run(int(fp64), int(GP), int(C_), C.byref(mh), C.byref(mp), x.ctypes.data_as(C.c_void_p), n,
                   y.ctypes.data_as(C.c_void_p), m, C.c_double(params.threshold), int(mask),
                   dense.ctypes.data_as(C.c_void_p), lz, C.byref(dist))
    r = EmuResult()
    r.code, r.P, r.dist = rc, dense, dist.value
    ln2 = math.log(2.0)
    ch = params.hmm.log_ins[x].sum() + params.hmm.log_ins[y].sum()
    cp = params.pf.log_ins[x].sum() + params.pf.log_ins[y].sum()
    r.logZ = np.array([lz[0] * ln2 + ch, lz[1] * ln2 + ch, lz[2] * ln2 + cp, lz[3] * ln2 + cp])
    nnz = L.emu_csr_nnz()
    r.row_ptr = np.zeros(n + 1, dtype=np.int32)
    r.rows, r.cols, r.vals = np.zeros(nnz, np.int32), np.zeros(nnz, np.int32), np.zeros(nnz, np.float32)
    L.emu_csr_get(r.row_ptr.ctypes.data_as(C.c_void_p), r.rows.ctypes.data_as(C.c_void_p),
                  r.cols.ctypes.data_as(C.c_void_p), r.vals.ctypes.data_as(C.c_void_p))
    return r
