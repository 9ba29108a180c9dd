"""Thin ctypes binding over libqp.so (include/qp.h). Argument marshalling only: every step of the hot path
(schedule, forward, backward, combine, sparsify, expected accuracy) runs in the CUDA kernels of csrc/.

PyTorch is used for device memory and streams only. There is no CPU fallback: importing this module raises if
libqp.so has not been built (python -m paper_1512_07437_b200.build), and calling it without a CUDA device fails.
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqp.so")

QP_OK = 0
ERR = {"INVALID_ARG": -1, "BAD_RESIDUE": -2, "EMPTY_SEQUENCE": -3, "BAD_PAIR": -4, "WORKSPACE_TOO_SMALL": -5,
       "NNZ_CAPACITY": -6, "CUDA": -7, "RANGE": -8, "STATIC_LIMIT": -9}
GUIDE_TREE_STATIC_MAX_K = 1024
QP_FP32, QP_FP64 = 0, 1
FLAG_SYNC_STATUS, FLAG_NO_REFINE, FLAG_NO_POLLERS = 1, 2, 4
NUM_CLASSES = 22

EXPORTS = ["qp_workspace_bytes", "qp_posteriors", "qp_posteriors_budgeted", "qp_guide_tree", "qp_guide_tree_workspace_bytes", "qp_last_launch_count", "qp_status_string", "qp_version",
           "qp_set_profile", "qp_get_profile", "qp_get_profile_classes", "qp_shutdown",
           "qp_consistency", "qp_consistency_workspace_bytes", "qp_consistency_passes", "qp_last_tau_curve", "qp_measure_peaks",
           "qp_posteriors_host", "qp_posteriors_host_workspace_bytes", "qp_guide_tree_static"]


class QpError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__(f"libqp: {status_string(code)} ({code}) {msg}")


class _Model(C.Structure):
    _fields_ = [("n_ins", C.c_int32), ("alphabet", C.c_int32),
                ("log_match", C.POINTER(C.c_double)), ("log_ins", C.POINTER(C.c_double)),
                ("t_MM", C.c_double), ("t_MI", C.c_double * 2), ("t_II", C.c_double * 2), ("t_IM", C.c_double * 2),
                ("init_M", C.c_double), ("init_I", C.c_double * 2), ("end_M", C.c_double), ("end_I", C.c_double * 2)]


class _Params(C.Structure):
    _fields_ = [("hmm", _Model), ("pf", _Model), ("threshold", C.c_double), ("precision", C.c_int32),
                ("flags", C.c_int32), ("refine_below", C.c_double)]


class _Output(C.Structure):
    _fields_ = [("pair_row_base", C.c_void_p), ("pair_nnz_base", C.c_void_p), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("val", C.c_void_p), ("nnz_capacity", C.c_int64), ("dist", C.c_void_p),
                ("dense_P", C.c_void_p), ("logZ", C.c_void_p), ("status", C.c_void_p)]


class _Csr(C.Structure):
    _fields_ = [("pair_row_base", C.c_void_p), ("pair_nnz_base", C.c_void_p), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("val", C.c_void_p)]


class _CsrOut(C.Structure):
    _fields_ = [("pair_nnz_base", C.c_void_p), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p), ("val", C.c_void_p),
                ("nnz_capacity", C.c_int64), ("relaxations", C.c_void_p), ("status", C.c_void_p)]


class _ConsParams(C.Structure):
    _fields_ = [("T", C.c_int32), ("f", C.c_int32), ("h", C.c_double), ("max_relax", C.c_int32), ("reserved", C.c_int32),
                ("threshold", C.c_double)]


class _HostOutput(C.Structure):
    _fields_ = [("pair_row_base", C.c_void_p), ("pair_nnz_base", C.c_void_p), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("val", C.c_void_p), ("nnz_capacity", C.c_int64), ("dist", C.c_void_p),
                ("col_idx16", C.c_void_p),
                ("beta_guess", C.c_double), ("status", C.c_int32 * 4), ("batches", C.c_int32), ("reserved", C.c_int32),
                ("h2d_bytes", C.c_int64), ("d2h_bytes", C.c_int64)]


class _Peaks(C.Structure):
    _fields_ = [("sms", C.c_int32), ("reserved", C.c_int32), ("ffma_per_s", C.c_double), ("ffma2_fma_per_s", C.c_double),
                ("mufu_per_s", C.c_double), ("warp_instr_per_s", C.c_double)]


SEL = {"max": 0, "min": 1, "sum": 2}


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1512_07437_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.qp_workspace_bytes.restype = C.c_int
    L.qp_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.POINTER(_Params), C.c_int64,
                                     C.c_int, C.c_size_t, C.POINTER(C.c_size_t)]
    L.qp_posteriors.restype = C.c_int
    L.qp_posteriors.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.POINTER(_Params),
                                C.c_void_p, C.c_size_t, C.POINTER(_Output), C.c_void_p]
    L.qp_posteriors_budgeted.restype = C.c_int
    L.qp_posteriors_budgeted.argtypes = L.qp_posteriors.argtypes + [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    L.qp_guide_tree_workspace_bytes.restype = C.c_size_t
    L.qp_guide_tree_workspace_bytes.argtypes = [C.c_int32]
    L.qp_guide_tree.restype = C.c_int
    L.qp_guide_tree.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_size_t, C.c_void_p]
    L.qp_guide_tree_static.restype = C.c_int
    L.qp_guide_tree_static.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p]
    L.qp_last_launch_count.restype = C.c_int
    L.qp_status_string.restype = C.c_char_p
    L.qp_status_string.argtypes = [C.c_int]
    L.qp_version.restype = C.c_char_p
    L.qp_set_profile.restype = None
    L.qp_set_profile.argtypes = [C.c_int]
    L.qp_get_profile.restype = C.c_int
    L.qp_get_profile.argtypes = [C.POINTER(C.c_float)]
    L.qp_get_profile_classes.restype = C.c_int
    L.qp_get_profile_classes.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_float)]
    L.qp_shutdown.restype = None
    L.qp_consistency_workspace_bytes.restype = C.c_int
    L.qp_consistency_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_int64, C.POINTER(C.c_size_t)]
    L.qp_consistency.restype = C.c_int
    L.qp_consistency.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.POINTER(_Csr), C.c_int64, C.c_void_p,
                                 C.POINTER(_ConsParams), C.c_void_p, C.c_size_t, C.POINTER(_CsrOut), C.c_void_p]
    L.qp_posteriors_host_workspace_bytes.restype = C.c_int
    L.qp_posteriors_host_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.POINTER(_Params), C.c_double,
                                                     C.POINTER(C.c_size_t)]
    L.qp_posteriors_host.restype = C.c_int
    L.qp_posteriors_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.POINTER(_Params), C.c_void_p,
                                     C.c_size_t, C.POINTER(_HostOutput), C.c_void_p]
    L.qp_measure_peaks.restype = C.c_int
    L.qp_measure_peaks.argtypes = [C.POINTER(_Peaks), C.c_void_p, C.c_size_t, C.c_void_p]
    L.qp_last_tau_curve.restype = C.c_int
    L.qp_last_tau_curve.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int64), C.c_int]
    L.qp_consistency_passes.restype = C.c_int
    L.qp_consistency_passes.argtypes = [C.c_int32]
    return L


_lib = _load()


def status_string(code: int) -> str:
    return _lib.qp_status_string(int(code)).decode()


def version() -> str:
    return _lib.qp_version().decode()


def last_launch_count() -> int:
    return int(_lib.qp_last_launch_count())


def shutdown() -> None:
    """qp_shutdown: release the calling thread's side streams and events (synchronise your streams first)."""
    _lib.qp_shutdown()


def set_profile(on: bool) -> None:
    _lib.qp_set_profile(int(bool(on)))


def get_profile():
    """Device ms of the last profiled call: dict(schedule, pair_kernels, refine, csr_place); `refine` = the fp64
    distance re-evaluation AND the CSR placement, which runs beside it; `csr_place` = what is left after their join
    (the status word). Sync the stream first."""
    ms = (C.c_float * 4)()
    r = _lib.qp_get_profile(ms)
    if r != QP_OK:
        raise QpError(r)
    return dict(schedule=ms[0], pair_kernels=ms[1], refine=ms[2], csr_place=ms[3])


def get_profile_classes():
    """[(class, start_ms, stop_ms)] of the class kernels of the last profiled call (relative to the fork);
    class = "C<stripe width>" for packed classes, "C<stripe width>xW<warps>" for split ones, "C<stripe width>mb" for
    the packed multi-block ones (one warp, the column blocks one after the other; fp32 naming)."""
    a, b = (C.c_float * NUM_CLASSES)(), (C.c_float * NUM_CLASSES)()
    r = _lib.qp_get_profile_classes(a, b)
    if r != QP_OK:
        raise QpError(r)
    names = ["C%d" % (c + 2) for c in range(15)] + ["C8xW4", "C12xW4", "C16xW4"] + ["C%dmb" % C for C in range(9, 13)]
    return [(names[c], round(a[c], 3), round(b[c], 3)) for c in range(NUM_CLASSES) if a[c] >= 0]


class CParams:
    """qp_params built from paper_1512_07437_b200.inputs.Params; keeps the host tables alive."""

    def __init__(self, params, precision="fp32", flags=FLAG_SYNC_STATUS, refine_below=0.0):
        self._keep = []
        s = _Params()
        for name in ("hmm", "pf"):
            m = getattr(params, name)
            lm = np.ascontiguousarray(m.log_match, dtype=np.float64)
            li = np.ascontiguousarray(m.log_ins, dtype=np.float64)
            self._keep += [lm, li]
            cm = getattr(s, name)
            cm.n_ins, cm.alphabet = int(m.n_ins), int(m.alphabet)
            cm.log_match = lm.ctypes.data_as(C.POINTER(C.c_double))
            cm.log_ins = li.ctypes.data_as(C.POINTER(C.c_double))
            cm.t_MM, cm.init_M, cm.end_M = float(m.t_MM), float(m.init_M), float(m.end_M)
            for f in ("t_MI", "t_II", "t_IM", "init_I", "end_I"):
                arr = getattr(cm, f)
                for g, v in enumerate(m.padded(f)):
                    arr[g] = v
        s.threshold = float(params.threshold)
        s.precision = QP_FP64 if precision in ("fp64", QP_FP64) else QP_FP32
        s.flags = int(flags)
        s.refine_below = float(refine_below)
        self.s = s

    @property
    def ref(self):
        return C.byref(self.s)


def min_workspace_bytes(h_offsets, k, h_pairs, cparams: CParams, nnz_capacity: int, want_dense=False) -> int:
    """The smallest workspace qp_posteriors accepts for this call (one scratch slot per class): the size that
    qp_workspace_bytes reports back when the budget it is given is too small."""
    h_offsets = np.ascontiguousarray(h_offsets, dtype=np.int64)
    h_pairs = np.ascontiguousarray(h_pairs, dtype=np.int32).reshape(-1, 2)
    out = C.c_size_t(0)
    r = _lib.qp_workspace_bytes(h_offsets.ctypes.data, int(k), h_pairs.ctypes.data, len(h_pairs), cparams.ref,
                                int(nnz_capacity), int(bool(want_dense)), 1, C.byref(out))
    if r not in (QP_OK, ERR["WORKSPACE_TOO_SMALL"]):
        raise QpError(r)
    return int(out.value)


def workspace_bytes(h_offsets, k, h_pairs, cparams: CParams, nnz_capacity: int, want_dense=False, budget=0) -> int:
    """qp_workspace_bytes: host-only query (numpy int64 offsets [k+1], int32 pairs [P,2])."""
    h_offsets = np.ascontiguousarray(h_offsets, dtype=np.int64)
    h_pairs = np.ascontiguousarray(h_pairs, dtype=np.int32).reshape(-1, 2)
    out = C.c_size_t(0)
    r = _lib.qp_workspace_bytes(h_offsets.ctypes.data, int(k), h_pairs.ctypes.data, len(h_pairs), cparams.ref,
                                int(nnz_capacity), int(bool(want_dense)), int(budget), C.byref(out))
    if r != QP_OK:
        raise QpError(r, f"(minimum workspace {out.value} bytes)" if r == ERR["WORKSPACE_TOO_SMALL"] else "")
    return int(out.value)


@dataclass
class Result:
    """Device tensors written by qp_posteriors (layout: include/qp.h `qp_output`)."""
    pair_row_base: object
    pair_nnz_base: object
    row_ptr: object
    col_idx: object
    val: object
    dist: object
    dense_P: object
    dense_off: object  # host numpy int64 [P+1] (only with want_dense)
    logZ: object
    status: object
    code: int
    launches: int
    tau_used: float = 0.0   # threshold the CSR was cut at (differs from the requested one in memory-limited mode)
    passes: int = 1

    def csr(self, p):
        """(row_ptr, col, val) of pair p as numpy arrays."""
        rb = self.pair_row_base[p:p + 2].tolist()
        nb = self.pair_nnz_base[p:p + 2].tolist()
        return (self.row_ptr[rb[0]:rb[1]].cpu().numpy(), self.col_idx[nb[0]:nb[1]].cpu().numpy(),
                self.val[nb[0]:nb[1]].cpu().numpy())


def alloc_outputs(device, max_pairs, max_rows_total, nnz_capacity, k, dist=None) -> Result:
    """Output tensors large enough for any call with P <= max_pairs, sum(n_p+1) <= max_rows_total (pass as `reuse=`)."""
    import torch
    i64, i32, f32 = torch.int64, torch.int32, torch.float32
    return Result(
        pair_row_base=torch.empty(max_pairs + 1, dtype=i64, device=device),
        pair_nnz_base=torch.empty(max_pairs + 1, dtype=i64, device=device),
        row_ptr=torch.empty(max(int(max_rows_total), 1), dtype=i32, device=device),
        col_idx=torch.empty(max(int(nnz_capacity), 1), dtype=i32, device=device),
        val=torch.empty(max(int(nnz_capacity), 1), dtype=f32, device=device),
        dist=dist if dist is not None else torch.zeros((k, k), dtype=f32, device=device),
        dense_P=None, dense_off=None, logZ=None, status=torch.zeros(4, dtype=i32, device=device), code=0, launches=0)


def posteriors(d_seqs, d_offsets, k, d_pairs, cparams: CParams, workspace, *, nnz_capacity, h_rows_total,
               want_dense_cells=0, want_logZ=False, dist=None, stream=None, check=True, reuse=None,
               budget_passes=0) -> Result:
    """qp_posteriors on torch CUDA tensors. `h_rows_total` = sum over pairs of (n_p + 1) (sizes row_ptr);
    `want_dense_cells` = sum n_p*m_p to also get the dense matrices (tests), 0 otherwise. `reuse` = a previous
    Result of the same shapes whose output tensors are written again instead of allocating new ones."""
    import torch

    dev = d_seqs.device
    P = int(d_pairs.shape[0])
    i64, i32, f32 = torch.int64, torch.int32, torch.float32
    o = _Output()
    if reuse is not None:
        t = dict(pair_row_base=reuse.pair_row_base, pair_nnz_base=reuse.pair_nnz_base, row_ptr=reuse.row_ptr,
                 col_idx=reuse.col_idx, val=reuse.val, dist=reuse.dist, dense_P=reuse.dense_P, logZ=reuse.logZ,
                 status=reuse.status)
    else:
        # fresh outputs are created (and zero-filled) on the stream the call runs on: torch would otherwise fill them
        # on its current stream, unordered with the kernels that write them
        with torch.cuda.stream(stream) if stream is not None else contextlib.nullcontext():
            t = dict(
                pair_row_base=torch.empty(P + 1, dtype=i64, device=dev),
                pair_nnz_base=torch.empty(P + 1, dtype=i64, device=dev),
                row_ptr=torch.empty(max(int(h_rows_total), 1), dtype=i32, device=dev),
                col_idx=torch.empty(max(int(nnz_capacity), 1), dtype=i32, device=dev),
                val=torch.empty(max(int(nnz_capacity), 1), dtype=f32, device=dev),
                dist=dist if dist is not None else torch.zeros((k, k), dtype=f32, device=dev),
                dense_P=torch.empty(int(want_dense_cells), dtype=f32, device=dev) if want_dense_cells else None,
                logZ=torch.empty((P, 4), dtype=torch.float64, device=dev) if want_logZ else None,
                status=torch.zeros(4, dtype=i32, device=dev),
            )
    for name, v in t.items():
        setattr(o, name, v.data_ptr() if v is not None else None)
    o.nnz_capacity = int(nnz_capacity)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    tau, passes = C.c_double(float(cparams.s.threshold)), C.c_int(1)
    with torch.cuda.device(dev):
        args = (d_seqs.data_ptr(), d_offsets.data_ptr(), int(k), d_pairs.data_ptr(), P, cparams.ref, workspace.data_ptr(),
                workspace.numel() * workspace.element_size(), C.byref(o), C.c_void_p(st.cuda_stream))
        if budget_passes:   # memory-limited mode: nnz_capacity is the budget, the threshold is raised until the CSR fits
            code = _lib.qp_posteriors_budgeted(*args, int(budget_passes), C.byref(tau), C.byref(passes))
        else:
            code = _lib.qp_posteriors(*args)
    res = Result(dense_off=None, code=int(code), launches=last_launch_count(), **t)
    res.tau_used, res.passes = float(tau.value), int(passes.value)
    if check and code != QP_OK:
        raise QpError(code)
    return res


def run_family(family, pairs, params, *, precision="fp32", want_dense=False, want_logZ=False, nnz_capacity=None,
               refine_below=0.0, flags=FLAG_SYNC_STATUS, device="cuda:0", budget=0, beta_guess=0.08) -> Result:
    """Convenience: host numpy family + pair list -> upload, size the workspace, call qp_posteriors, and retry
    once with the exact capacity if the CSR did not fit. Returns device tensors."""
    import torch

    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    L = family.lengths
    n, m = L[pairs[:, 0]], L[pairs[:, 1]]
    cells = int((n * m).sum()) if len(pairs) else 0
    rows_total = int((n + 1).sum()) if len(pairs) else 0
    cp = CParams(params, precision=precision, flags=flags, refine_below=refine_below)
    dev = torch.device(device)
    d_seqs = torch.from_numpy(np.ascontiguousarray(family.seqs)).to(dev)
    d_offs = torch.from_numpy(np.ascontiguousarray(family.offsets, dtype=np.int64)).to(dev)
    d_pairs = torch.from_numpy(pairs).to(dev)
    cap = int(nnz_capacity) if nnz_capacity is not None else int(beta_guess * cells) + 1024
    for attempt in range(2):
        wsb = workspace_bytes(family.offsets, family.k, pairs, cp, cap, want_dense, budget)
        ws = torch.empty(wsb, dtype=torch.uint8, device=dev)
        res = posteriors(d_seqs, d_offs, family.k, d_pairs, cp, ws, nnz_capacity=cap, h_rows_total=rows_total,
                         want_dense_cells=cells if want_dense else 0, want_logZ=want_logZ, check=False)
        if res.code == ERR["NNZ_CAPACITY"] and attempt == 0 and nnz_capacity is None:
            cap = int(res.pair_nnz_base[-1].item())
            continue
        if res.code != QP_OK:
            raise QpError(res.code)
        break
    if want_dense:
        res.dense_off = np.concatenate([[0], np.cumsum(n.astype(np.int64) * m.astype(np.int64))])
    return res


@dataclass
class GuideTree:
    """Device tensors written by qp_guide_tree (layout: include/qp.h)."""
    merge: object      # int32 [k-1, 2]
    height: object     # float32 [k-1]
    leaves: object     # int32 [2k-1]
    parent: object     # int32 [2k-1]
    treedist: object   # int32 [k, k] or None


def guide_tree(dist, want_treedist=True, stream=None, workspace=None) -> GuideTree:
    """qp_guide_tree on a k x k float32 CUDA tensor (the distance matrix of qp_posteriors): weighted UPGMA guide tree
    and, optionally, the tree-guided distances. Marshalling only; enqueued on the stream, not synchronised."""
    import torch
    assert dist.is_cuda and dist.dtype == torch.float32 and dist.dim() == 2 and dist.shape[0] == dist.shape[1]
    dist = dist.contiguous()
    k, dev = int(dist.shape[0]), dist.device
    i32 = torch.int32
    t = GuideTree(merge=torch.empty((max(k - 1, 0), 2), dtype=i32, device=dev),
                  height=torch.empty(max(k - 1, 0), dtype=torch.float32, device=dev),
                  leaves=torch.empty(2 * k - 1, dtype=i32, device=dev), parent=torch.empty(2 * k - 1, dtype=i32, device=dev),
                  treedist=torch.empty((k, k), dtype=i32, device=dev) if want_treedist else None)
    need = int(_lib.qp_guide_tree_workspace_bytes(k))
    ws = workspace if workspace is not None else torch.empty(need, dtype=torch.uint8, device=dev)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    with torch.cuda.device(dev):
        code = _lib.qp_guide_tree(dist.data_ptr(), k, t.merge.data_ptr(), t.height.data_ptr(), t.leaves.data_ptr(),
                                  t.parent.data_ptr(), t.treedist.data_ptr() if want_treedist else None, ws.data_ptr(),
                                  ws.numel(), C.c_void_p(st.cuda_stream))
    if code != QP_OK:
        raise QpError(code)
    t._ws = ws   # keep the workspace alive until the stream has run
    return t


def guide_tree_static(out: GuideTree, dist, stream=None) -> GuideTree:
    """qp_guide_tree_static: the guide tree of `dist` written into the tensors of `out`, with the merge loop's scratch in
    the array built into libqp.so instead of a workspace. For callers that cannot allocate device memory at the point of
    the call (all device memory owned by a host application, a loop that must not block in the driver, a fixed memory
    reservation on a shared GPU) -- which is why this wrapper creates no tensor either: `dist` (k x k float32,
    contiguous, CUDA) and every tensor of `out` (shapes of GuideTree for the same k; treedist may be None) are made by
    the caller beforehand. k <= GUIDE_TREE_STATIC_MAX_K, else QpError(STATIC_LIMIT). All calls on a device share the one
    scratch array: keep them on one stream, or order them, or they race. The first call per device resolves the array's
    address; make it outside stream capture. Enqueued on the stream, not synchronised."""
    import torch
    assert dist.is_cuda and dist.dtype == torch.float32 and dist.dim() == 2 and dist.shape[0] == dist.shape[1]
    assert dist.is_contiguous(), "no copy is made here: pass a contiguous matrix"
    k, dev = int(dist.shape[0]), dist.device
    assert out.leaves.numel() == 2 * k - 1 and out.parent.numel() == 2 * k - 1 and out.merge.numel() == 2 * max(k - 1, 0)
    assert out.height.numel() == max(k - 1, 0) and (out.treedist is None or out.treedist.numel() == k * k)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    with torch.cuda.device(dev):
        code = _lib.qp_guide_tree_static(dist.data_ptr(), k, out.merge.data_ptr(), out.height.data_ptr(),
                                         out.leaves.data_ptr(), out.parent.data_ptr(),
                                         out.treedist.data_ptr() if out.treedist is not None else None,
                                         C.c_void_p(st.cuda_stream))
    if code != QP_OK:
        raise QpError(code)
    return out


def last_tau_curve(max_bins: int = 128):
    """qp_last_tau_curve: (tau[b], count of kept values >= tau[b]) of the last memory-limited call, numpy arrays."""
    tau, cnt = (C.c_double * max_bins)(), (C.c_int64 * max_bins)()
    n = _lib.qp_last_tau_curve(tau, cnt, int(max_bins))
    if n < 0:
        raise QpError(n)
    return np.array(tau[:n]), np.array(cnt[:n], dtype=np.int64)


def measure_peaks(device="cuda:0") -> dict:
    """qp_measure_peaks: measured FFMA / FFMA2 / MUFU rates and the warp-instruction issue rate of the device."""
    import torch
    dev = torch.device(device)
    scratch = torch.empty(1 << 20, dtype=torch.uint8, device=dev)
    pk = _Peaks()
    with torch.cuda.device(dev):
        r = _lib.qp_measure_peaks(C.byref(pk), scratch.data_ptr(), scratch.numel(), C.c_void_p(torch.cuda.current_stream(dev).cuda_stream))
    if r != QP_OK:
        raise QpError(r)
    return dict(sms=pk.sms, ffma_per_s=pk.ffma_per_s, ffma2_fma_per_s=pk.ffma2_fma_per_s, mufu_per_s=pk.mufu_per_s,
                warp_instr_per_s=pk.warp_instr_per_s)


def consistency_passes(k: int) -> int:
    """qp_consistency_passes: the paper's rule, 2 transformations for k < 50, 1 otherwise."""
    return int(_lib.qp_consistency_passes(int(k)))


def consistency(d_offsets, k, d_pairs, csr, treedist, *, h_offsets, h_pairs, nnz=None, T=200, f="max", h=3.0,
                max_relax=200, threshold=0.01, stream=None, workspace=None, check=True) -> Result:
    """qp_consistency (stage III, selective consistency) on torch CUDA tensors. `csr` = anything with the members
    pair_row_base / pair_nnz_base / row_ptr / col_idx / val (a Result of `posteriors` or of a previous call);
    `treedist` = int32 k x k (GuideTree.treedist). Marshalling only. Returns a Result whose pair_row_base is the
    input's (rows do not change), with `.relaxations` (int32 [P]) attached. Synchronises once to read the status
    (and, if `nnz` is not given, once to read the input's entry count)."""
    import torch
    dev = d_pairs.device
    P = int(d_pairs.shape[0])
    if nnz is None:
        nnz = int(csr.pair_nnz_base[P].item()) if P else 0
    h_offsets = np.ascontiguousarray(h_offsets, dtype=np.int64)
    h_pairs = np.ascontiguousarray(h_pairs, dtype=np.int32).reshape(-1, 2)
    need = C.c_size_t(0)
    r = _lib.qp_consistency_workspace_bytes(h_offsets.ctypes.data, int(k), h_pairs.ctypes.data, P, int(nnz), C.byref(need))
    if r != QP_OK:
        raise QpError(r)
    ws = workspace if workspace is not None else torch.empty(max(int(need.value), 256), dtype=torch.uint8, device=dev)
    i64, i32, f32 = torch.int64, torch.int32, torch.float32
    rows_total = int(csr.row_ptr.numel())
    # the zero-filled outputs are created, and the status is read back, on the stream the call runs on
    on_stream = (lambda: torch.cuda.stream(stream)) if stream is not None else contextlib.nullcontext
    with on_stream():
        out = Result(pair_row_base=csr.pair_row_base, pair_nnz_base=torch.empty(P + 1, dtype=i64, device=dev),
                     row_ptr=torch.empty(max(rows_total, 1), dtype=i32, device=dev),
                     col_idx=torch.empty(max(int(nnz), 1), dtype=i32, device=dev),
                     val=torch.empty(max(int(nnz), 1), dtype=f32, device=dev), dist=None, dense_P=None, dense_off=None,
                     logZ=None, status=torch.zeros(4, dtype=i32, device=dev), code=0, launches=9)
        out.relaxations = torch.zeros(max(P, 1), dtype=i32, device=dev)
    ci = _Csr(csr.pair_row_base.data_ptr(), csr.pair_nnz_base.data_ptr(), csr.row_ptr.data_ptr(), csr.col_idx.data_ptr(),
              csr.val.data_ptr())
    co = _CsrOut(out.pair_nnz_base.data_ptr(), out.row_ptr.data_ptr(), out.col_idx.data_ptr(), out.val.data_ptr(), int(nnz),
                 out.relaxations.data_ptr(), out.status.data_ptr())
    prm = _ConsParams(int(T), SEL[f] if isinstance(f, str) else int(f), float(h), int(max_relax), 0, float(threshold))
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    with torch.cuda.device(dev):
        code = _lib.qp_consistency(d_offsets.data_ptr(), int(k), d_pairs.data_ptr(), P, C.byref(ci), int(nnz),
                                   treedist.data_ptr(), C.byref(prm), ws.data_ptr(), ws.numel(), C.byref(co),
                                   C.c_void_p(st.cuda_stream))
    out._ws = ws
    if code == QP_OK and check:
        with on_stream():
            code = int(out.status[0].item())      # synchronises
    out.code = int(code)
    if check and code != QP_OK:
        raise QpError(code)
    return out


class HostCall:
    """qp_posteriors_host: the posterior stage on HOST buffers (pinned torch CPU tensors), one C call per family.
    Allocates the pinned inputs / outputs and the device workspace once; `run()` may be called again and again.
    Marshalling only: batching, copies and stream ordering happen inside libqp.so (csrc/qp_host.cu)."""

    def __init__(self, family, pairs, params, *, device="cuda:0", beta_guess=0.05, nnz_capacity=None, workspace_bytes=None,
                 precision="fp32", flags=0, compact_cols=False):
        import torch
        self.torch = torch
        self.dev = torch.device(device)
        self.k = int(family.k)
        pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        self.P = len(pairs)
        L = family.lengths
        n, m = L[pairs[:, 0]].astype(np.int64), L[pairs[:, 1]].astype(np.int64)
        self.cells = int((n * m).sum())
        rows_total = int((n + 1).sum())
        self.cp = CParams(params, precision=precision, flags=flags)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        self.h_seqs, self.h_offs, self.h_pairs = pin(family.seqs), pin(family.offsets.astype(np.int64)), pin(pairs)
        cap = int(nnz_capacity) if nnz_capacity is not None else int(1.2 * beta_guess * self.cells) + 4096
        e = lambda size, dt: torch.empty(max(int(size), 1), dtype=dt).pin_memory()
        self.pair_row_base, self.pair_nnz_base = e(self.P + 1, torch.int64), e(self.P + 1, torch.int64)
        # compact_cols: the columns come back as 16-bit values (col_idx16, uint16) instead of int32 (col_idx)
        self.row_ptr, self.val = e(rows_total, torch.int32), e(cap, torch.float32)
        self.col_idx = None if compact_cols else e(cap, torch.int32)
        self.col_idx16 = e(cap, torch.int16).view(torch.uint16) if compact_cols else None   # pinned as int16, read as uint16
        self.dist = torch.empty((self.k, self.k), dtype=torch.float32).pin_memory()
        self.cap, self.beta_guess = cap, float(beta_guess)
        need = C.c_size_t(0)
        r = _lib.qp_posteriors_host_workspace_bytes(self.h_offs.data_ptr(), self.k, self.h_pairs.data_ptr(), self.P, self.cp.ref,
                                                    self.beta_guess, C.byref(need))
        if r != QP_OK:
            raise QpError(r)
        self.ws = torch.empty(int(workspace_bytes) if workspace_bytes else max(int(need.value), 256), dtype=torch.uint8, device=self.dev)
        self.out = _HostOutput()

    def run(self, stream=None, check=True):
        """One call. Returns self (pinned tensors pair_row_base, pair_nnz_base, row_ptr, col_idx, val, dist are filled;
        .nnz, .batches, .h2d_bytes, .d2h_bytes, .code, .refined are set)."""
        torch = self.torch
        o = self.out
        o.pair_row_base, o.pair_nnz_base, o.row_ptr = self.pair_row_base.data_ptr(), self.pair_nnz_base.data_ptr(), self.row_ptr.data_ptr()
        o.col_idx = self.col_idx.data_ptr() if self.col_idx is not None else None
        o.col_idx16 = self.col_idx16.data_ptr() if self.col_idx16 is not None else None
        o.val, o.nnz_capacity, o.dist = self.val.data_ptr(), self.cap, self.dist.data_ptr()
        o.beta_guess = self.beta_guess
        st = stream if stream is not None else torch.cuda.current_stream(self.dev)
        with torch.cuda.device(self.dev):
            code = _lib.qp_posteriors_host(self.h_seqs.data_ptr(), self.h_offs.data_ptr(), self.k, self.h_pairs.data_ptr(), self.P,
                                           self.cp.ref, self.ws.data_ptr(), self.ws.numel(), C.byref(o), C.c_void_p(st.cuda_stream))
        self.code, self.batches = int(code), int(o.batches)
        self.h2d_bytes, self.d2h_bytes, self.refined = int(o.h2d_bytes), int(o.d2h_bytes), int(o.status[3])
        self.nnz = int(self.pair_nnz_base[self.P].item()) if self.P else 0
        if check and code != QP_OK:
            raise QpError(code, f"(pair {o.status[1]})")
        return self
