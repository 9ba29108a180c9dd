"""Host-buffer front end of qp_posteriors: stream a family's pair list through the GPU in batches.

BASELINE.json configs[3]: "memory-budgeted by streaming pair batches". The caller's data lives in HOST memory
(pinned): sequences, offsets and the pair list go host -> device, the k x k distance matrix and the whole CSR
(pair_row_base, pair_nnz_base, row_ptr, col_idx, val) come back device -> host, batch by batch. Two batches are in
flight: while batch b's CSR travels back over PCIe on its slot's copy stream, batch b+1's kernels run on the compute
stream, so the wall time of a family is max(compute, copy) instead of their sum. (The C library has the same driver
as one call: qp_posteriors_host / qp.HostCall; this class is the generator variant that hands every batch out as soon
as it is in host memory.) Every step of the computation still runs inside
qp_posteriors (CUDA); this module only moves buffers and orders streams.

    s = HostStreamer(family, pairs, params)          # allocates device workspaces + pinned staging once
    for batch in s.run():                             # batch.lo, batch.hi, batch.row_base, batch.nnz_base, batch.row_ptr, batch.col, batch.val
        consume(batch)                                # valid until the next-but-one batch is produced
    s.dist                                            # pinned k x k float32, complete after run()
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import qp


@dataclass
class HostBatch:
    """One batch of pairs [lo, hi) with its CSR in pinned host memory (views into the streamer's staging buffers)."""
    lo: int
    hi: int
    row_base: object   # int64 [hi-lo+1]
    nnz_base: object   # int64 [hi-lo+1]
    row_ptr: object    # int32 [sum(n_p+1)]
    col: object        # int32 [nnz]
    val: object        # float32 [nnz]


class HostStreamer:
    def __init__(self, family, pairs, params, device="cuda:0", batch_cells=None, beta_guess=0.05, precision="fp32"):
        import torch
        self.torch = torch
        self.dev = torch.device(device)
        self.fam = family
        self.pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        L = family.lengths
        self.n = L[self.pairs[:, 0]].astype(np.int64)
        m = L[self.pairs[:, 1]].astype(np.int64)
        cells = self.n * m
        self.cells = int(cells.sum())
        if batch_cells is None:   # at least four batches (so that copies can overlap kernels), at most ~2 GB of CSR each
            batch_cells = min(6.0e9, max(4.0e8, self.cells / 4.0))
        # batches of about batch_cells cells (about 0.05 * batch_cells CSR entries each)
        bounds, acc = [0], 0
        for p in range(len(self.pairs)):
            acc += int(cells[p])
            if acc >= batch_cells:
                bounds.append(p + 1)
                acc = 0
        if bounds[-1] != len(self.pairs):
            bounds.append(len(self.pairs))
        self.bounds = bounds
        nb = len(bounds) - 1
        self.rows = [int((self.n[bounds[b]:bounds[b + 1]] + 1).sum()) for b in range(nb)]
        max_cells = max(int(cells[bounds[b]:bounds[b + 1]].sum()) for b in range(nb)) if nb else 0
        max_rows = max(self.rows) if nb else 1
        max_pairs = max(bounds[b + 1] - bounds[b] for b in range(nb)) if nb else 1
        self.cap = int(beta_guess * max_cells) + 4096
        self.cp = qp.CParams(params, precision=precision, flags=0)   # no sync inside the call: status is read with the CSR sizes
        i64, i32, f32 = torch.int64, torch.int32, torch.float32
        self.h_seqs = torch.from_numpy(np.ascontiguousarray(family.seqs)).pin_memory()
        self.h_offs = torch.from_numpy(np.ascontiguousarray(family.offsets, dtype=np.int64)).pin_memory()
        self.h_pairs = torch.from_numpy(self.pairs).pin_memory()
        self.dist = torch.empty((family.k, family.k), dtype=f32).pin_memory()
        self.d_dist = torch.zeros((family.k, family.k), dtype=f32, device=self.dev)
        self.max_pairs, self.max_rows = max_pairs, max_rows
        self.comp = torch.cuda.Stream(self.dev)     # every batch's kernels, in order
        self.slots = []
        for _ in range(2):   # two batches in flight
            sl = dict(
                stream=torch.cuda.Stream(self.dev),
                d_pairs=torch.empty((max_pairs, 2), dtype=i32, device=self.dev),
                h_rp=torch.empty(max_rows, dtype=i32).pin_memory(),
                h_rb=torch.empty(max_pairs + 1, dtype=i64).pin_memory(),
                h_nb=torch.empty(max_pairs + 1, dtype=i64).pin_memory(),
                h_status=torch.empty(4, dtype=i32).pin_memory(),
                sized=torch.cuda.Event(), done=torch.cuda.Event(),
            )
            self._size_slot(sl, self.cap)
            self.slots.append(sl)
        self.h2d_bytes = self.d2h_bytes = 0
        self.launches = 0
        self.retries = 0

    def _size_slot(self, sl, cap):
        """(Re)allocate what depends on the CSR capacity of a slot: workspace (it holds the staging pool), device CSR,
        pinned CSR."""
        torch = self.torch
        nb = len(self.bounds) - 1
        wsb = max((qp.workspace_bytes(self.fam.offsets, self.fam.k, self.pairs[self.bounds[b]:self.bounds[b + 1]], self.cp, cap)
                   for b in range(nb)), default=256)
        for key in ("ws", "res", "h_col", "h_val"):
            sl.pop(key, None)
        sl["cap"] = int(cap)
        sl["ws"] = torch.empty(wsb, dtype=torch.uint8, device=self.dev)
        sl["res"] = qp.alloc_outputs(self.dev, self.max_pairs, self.max_rows, cap, self.fam.k, dist=self.d_dist)
        sl["h_col"] = torch.empty(cap, dtype=torch.int32).pin_memory()
        sl["h_val"] = torch.empty(cap, dtype=torch.float32).pin_memory()

    def _enqueue(self, b, d_seqs, d_offs):
        """H2D of the batch's pairs, the call, D2H of the sizes and the status on the ONE compute stream (two calls with
        their persistent kernels side by side starve each other's short tail kernels); the other small arrays on the
        slot's copy stream."""
        torch = self.torch
        s = self.slots[b % 2]
        lo, hi = self.bounds[b], self.bounds[b + 1]
        self.comp.wait_event(s["done"])            # the slot's previous CSR has left the device
        with torch.cuda.stream(self.comp):
            s["d_pairs"][: hi - lo].copy_(self.h_pairs[lo:hi], non_blocking=True)
            r = qp.posteriors(d_seqs, d_offs, self.fam.k, s["d_pairs"][: hi - lo], self.cp, s["ws"], nnz_capacity=s["cap"],
                              h_rows_total=self.rows[b], stream=self.comp, check=True, reuse=s["res"])
            res = s["res"]
            s["h_nb"][: hi - lo + 1].copy_(res.pair_nnz_base[: hi - lo + 1], non_blocking=True)
            s["h_status"].copy_(res.status, non_blocking=True)
            s["sized"].record(self.comp)
        s["stream"].wait_event(s["sized"])
        with torch.cuda.stream(s["stream"]):
            s["h_rb"][: hi - lo + 1].copy_(res.pair_row_base[: hi - lo + 1], non_blocking=True)
            s["h_rp"][: self.rows[b]].copy_(res.row_ptr[: self.rows[b]], non_blocking=True)
        self.launches += r.launches
        self.h2d_bytes += 8 * (hi - lo)

    def _collect(self, b, d_seqs, d_offs):
        """Wait for the batch's sizes, then D2H of exactly nnz entries of col/val on the slot's stream. A batch whose
        CSR did not fit the slot's capacity (denser than beta_guess) is run again, once, in a slot grown to the entry
        count the failed call reported; the batches already handed out are not affected."""
        torch = self.torch
        s = self.slots[b % 2]
        lo, hi = self.bounds[b], self.bounds[b + 1]
        s["sized"].synchronize()
        code = int(s["h_status"][0].item())
        if code == qp.ERR["NNZ_CAPACITY"]:
            need = int(s["h_nb"][hi - lo].item())          # pair_nnz_base[P] = entries required
            self._size_slot(s, need + need // 16 + 4096)
            self.retries += 1
            self._enqueue(b, d_seqs, d_offs)
            s["sized"].synchronize()
            code = int(s["h_status"][0].item())
        if code != qp.QP_OK:
            raise qp.QpError(code, f"(batch {b}, pairs {lo}..{hi})")
        nz = int(s["h_nb"][hi - lo].item())
        with torch.cuda.stream(s["stream"]):
            s["h_col"][:nz].copy_(s["res"].col_idx[:nz], non_blocking=True)
            s["h_val"][:nz].copy_(s["res"].val[:nz], non_blocking=True)
            s["done"].record(s["stream"])
        self.d2h_bytes += 16 * (hi - lo + 1) + 16 + 4 * self.rows[b] + 8 * nz
        return nz

    def run(self):
        """Generator over HostBatch. Batch b is yielded once its CSR is in host memory; batch b+1 is computing meanwhile."""
        torch = self.torch
        nb = len(self.bounds) - 1
        main = torch.cuda.current_stream(self.dev)
        d_seqs = self.h_seqs.to(self.dev, non_blocking=True)
        d_offs = self.h_offs.to(self.dev, non_blocking=True)
        up = torch.cuda.Event()
        up.record(main)
        self.h2d_bytes += self.h_seqs.numel() + 8 * self.h_offs.numel()
        self.comp.wait_event(up)
        if nb:
            self._enqueue(0, d_seqs, d_offs)
        for b in range(nb):
            # batch b is computing. Batch b-1 (the other slot) was handed out by the previous `yield` and the caller
            # has come back for more, so that slot is free: start batch b+1 in it before waiting for batch b.
            if b + 1 < nb:
                self._enqueue(b + 1, d_seqs, d_offs)
            nz = self._collect(b, d_seqs, d_offs)   # D2H of batch b's CSR overlaps batch b+1's kernels
            s = self.slots[b % 2]
            lo, hi = self.bounds[b], self.bounds[b + 1]
            s["done"].synchronize()
            if b == nb - 1:
                break
            yield HostBatch(lo, hi, s["h_rb"][: hi - lo + 1], s["h_nb"][: hi - lo + 1], s["h_rp"][: self.rows[b]],
                            s["h_col"][:nz], s["h_val"][:nz])
        main.wait_stream(self.comp)
        for sl in self.slots:
            main.wait_stream(sl["stream"])
        self.dist.copy_(self.d_dist, non_blocking=True)
        main.synchronize()
        self.d2h_bytes += 4 * self.fam.k * self.fam.k
        if nb:   # the last batch goes out once the distance matrix is complete too
            yield HostBatch(lo, hi, s["h_rb"][: hi - lo + 1], s["h_nb"][: hi - lo + 1], s["h_rp"][: self.rows[nb - 1]],
                            s["h_col"][:nz], s["h_val"][:nz])
