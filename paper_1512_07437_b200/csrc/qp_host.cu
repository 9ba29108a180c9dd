// qp_host.cu -- qp_posteriors_host: the posterior stage on HOST buffers (include/qp.h).
//
// BASELINE.json configs[3]: "memory-budgeted by streaming pair batches". The caller's data lives in host memory;
// the pair list is cut into batches that fit the device workspace twice, and two batches are in flight: while batch
// b's CSR travels back over PCIe on the slot's copy stream, batch b+1's kernels run on the compute stream, so the wall
// time of a family is max(compute, copy) instead of their sum. Every step of the computation runs inside qp_posteriors (this file
// only plans batches, moves buffers and orders streams; it is written against the public C ABI; its one kernel
// narrows the column indices to 16 bits when the caller asks for the compact form).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <vector>

#include "qp.h"

namespace {

inline int64_t al256(int64_t v) { return (v + 255) & ~(int64_t)255; }

// columns as 16-bit values for the trip over PCIe (QP_MAX_LEN = 65535: lossless); the count is read on the device
// (a batch whose CSR did not fit reports the size it NEEDS there: never walk past the slot's capacity)
__global__ void k_narrow_cols(const int32_t* __restrict__ col, const int64_t* __restrict__ count, int64_t cap,
                              uint16_t* __restrict__ col16) {
    const int64_t n = *count < cap ? *count : cap;
    for (int64_t q = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) * 2; q < n; q += (int64_t)gridDim.x * blockDim.x * 2) {
        if (q + 1 < n) *(ushort2*)(col16 + q) = make_ushort2((unsigned short)col[q], (unsigned short)col[q + 1]);
        else col16[q] = (uint16_t)col[q];
    }
}

struct Batch {
    int64_t lo, hi;        // pairs [lo, hi)
    int64_t cells, rows;   // sum n*m, sum (n+1)
};

struct Slot {              // device buffers of one batch in flight + its stream
    cudaStream_t st = nullptr;
    cudaEvent_t sized = nullptr, done = nullptr;
    char* base = nullptr;
    int32_t* pairs = nullptr;
    int64_t *row_base = nullptr, *nnz_base = nullptr;
    int32_t *row_ptr = nullptr, *col = nullptr, *status = nullptr;
    uint16_t* col16 = nullptr;
    float* val = nullptr;
    char* ws = nullptr;
    int64_t ws_bytes = 0, cap = 0;
    // pinned staging of the small per-batch results (sizes and status), owned by the call
    int64_t* h_last = nullptr;   // [1] nnz of the batch
    int32_t* h_status = nullptr; // [4]
    Batch cur{0, 0, 0, 0};
    int64_t out_nnz0 = 0;        // where the batch's entries go in the caller's col_idx / val
};

struct SlotPlan {
    int64_t max_pairs, max_rows, cap, ws_bytes, total;
};

// bytes of one slot for batches of at most these sizes
SlotPlan plan_slot(int64_t max_pairs, int64_t max_rows, int64_t cap, int64_t ws_bytes) {
    SlotPlan p{max_pairs, max_rows, cap, ws_bytes, 0};
    p.total = al256(max_pairs * 8) + 2 * al256((max_pairs + 1) * 8) + al256(max_rows * 4) + 2 * al256(cap * 4) + al256(cap * 2) +
              256 + al256(ws_bytes);
    return p;
}

}  // namespace

extern "C" int qp_posteriors_host_workspace_bytes(const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P,
                                                  const qp_params* params, double beta_guess, size_t* out_bytes) {
    if (!h_offsets || (!h_pairs && P > 0) || !params || !out_bytes || k < 0 || P < 0) return QP_ERR_INVALID_ARG;
    const double beta = beta_guess > 0.0 ? beta_guess : 0.05;
    int64_t total_cells = 0;
    std::vector<int64_t> cells(P), rows(P);
    for (int64_t p = 0; p < P; ++p) {
        const int x = h_pairs[2 * p], y = h_pairs[2 * p + 1];
        if (x < 0 || y < 0 || x >= k || y >= k || x == y) return QP_ERR_BAD_PAIR;
        const int64_t n = h_offsets[x + 1] - h_offsets[x], m = h_offsets[y + 1] - h_offsets[y];
        if (n < 1 || m < 1 || n > QP_MAX_LEN || m > QP_MAX_LEN) return QP_ERR_EMPTY_SEQUENCE;
        cells[p] = n * m;
        rows[p] = n + 1;
        total_cells += cells[p];
    }
    // the batch size qp_posteriors_host aims at first: a quarter of the family, between 4e8 and 6e9 cells
    const double target = std::min(6.0e9, std::max(4.0e8, (double)total_cells / 4.0));
    int64_t max_pairs = 0, max_rows = 0, max_cells = 0, lo = 0, c = 0, r = 0;
    size_t worst = 0;
    qp_params prm = *params;
    std::vector<std::pair<int64_t, int64_t>> bounds;
    for (int64_t p = 0; p < P; ++p) {
        c += cells[p];
        r += rows[p];
        if ((double)c >= target || p + 1 == P) {
            bounds.push_back({lo, p + 1});
            max_pairs = std::max(max_pairs, p + 1 - lo);
            max_rows = std::max(max_rows, r);
            max_cells = std::max(max_cells, c);
            lo = p + 1;
            c = r = 0;
        }
    }
    const int64_t cap = (int64_t)(beta * (double)max_cells) + 4096;
    for (auto& b : bounds) {
        size_t wsb = 0;
        const int rr = qp_workspace_bytes(h_offsets, k, h_pairs + 2 * b.first, b.second - b.first, &prm, cap, 0, 0, &wsb);
        if (rr != QP_OK) return rr;
        worst = std::max(worst, wsb);
    }
    const int64_t seq_bytes = h_offsets[k] - h_offsets[0];
    const int64_t common = al256(seq_bytes) + al256((int64_t)(k + 1) * 8) + al256((int64_t)k * k * 4);
    *out_bytes = (size_t)(common + 2 * plan_slot(max_pairs, max_rows, cap, (int64_t)worst).total);
    return QP_OK;
}

extern "C" int qp_posteriors_host(const uint8_t* h_seqs, const int64_t* h_offsets, int32_t k, const int32_t* h_pairs,
                                  int64_t P, const qp_params* params, void* d_workspace, size_t workspace_bytes,
                                  qp_host_output* out, void* cuda_stream) {
    if (!out || !params || !h_offsets || k < 0 || P < 0 || (P > 0 && (!h_seqs || !h_pairs || !d_workspace))) return QP_ERR_INVALID_ARG;
    if (!out->pair_row_base || !out->pair_nnz_base || (P > 0 && (!out->row_ptr || !out->dist))) return QP_ERR_INVALID_ARG;
    if (out->nnz_capacity < 0 || (out->nnz_capacity > 0 && ((!out->col_idx && !out->col_idx16) || !out->val))) return QP_ERR_INVALID_ARG;
    if (((uintptr_t)d_workspace & 255) != 0) return QP_ERR_INVALID_ARG;
    out->h2d_bytes = out->d2h_bytes = 0;
    out->batches = 0;
    out->status[0] = out->status[1] = out->status[2] = out->status[3] = 0;
    out->pair_row_base[0] = out->pair_nnz_base[0] = 0;
    if (P == 0) return QP_OK;
    cudaStream_t main = (cudaStream_t)cuda_stream;
    const double beta = out->beta_guess > 0.0 ? out->beta_guess : 0.05;

    // ---- host-side plan: per-pair sizes, prefix of rows, batches ---------------------------------------------------
    std::vector<int64_t> cells(P);
    int64_t total_cells = 0;
    for (int64_t p = 0; p < P; ++p) {
        const int x = h_pairs[2 * p], y = h_pairs[2 * p + 1];
        if (x < 0 || y < 0 || x >= k || y >= k || x == y) {
            out->status[0] = QP_ERR_BAD_PAIR;
            out->status[1] = (int32_t)p;
            return QP_ERR_BAD_PAIR;
        }
        const int64_t n = h_offsets[x + 1] - h_offsets[x], m = h_offsets[y + 1] - h_offsets[y];
        if (n < 1 || m < 1 || n > QP_MAX_LEN || m > QP_MAX_LEN) {
            out->status[0] = QP_ERR_EMPTY_SEQUENCE;
            out->status[1] = (int32_t)p;
            return QP_ERR_EMPTY_SEQUENCE;
        }
        cells[p] = n * m;
        total_cells += cells[p];
        out->pair_row_base[p + 1] = out->pair_row_base[p] + n + 1;
    }
    const int64_t seq_bytes = h_offsets[k] - h_offsets[0];
    const int64_t common = al256(seq_bytes) + al256((int64_t)(k + 1) * 8) + al256((int64_t)k * k * 4);
    qp_params prm = *params;
    prm.flags &= ~QP_FLAG_SYNC_STATUS;   // the batches' kernels run one call after the other on one stream
    // no pollers: the waiting fp64 kernels of batch b would sit in front of batch b + 1's kernels in the hardware queues
    // the calls share (measured on configs[3]: 341 ms per family without, 380 ms with them)
    prm.flags |= QP_FLAG_NO_POLLERS;

    std::vector<Batch> batches;
    SlotPlan sp{0, 0, 0, 0, 0};
    // at least four batches when the family is large (so that copies overlap kernels), at most ~6e9 cells each;
    // shrink until two slots fit the workspace
    double target = std::min(6.0e9, std::max(4.0e8, (double)total_cells / 4.0));
    for (int attempt = 0; attempt < 40; ++attempt) {
        batches.clear();
        Batch b{0, 0, 0, 0};
        for (int64_t p = 0; p < P; ++p) {
            b.cells += cells[p];
            b.rows += out->pair_row_base[p + 1] - out->pair_row_base[p];
            b.hi = p + 1;
            if ((double)b.cells >= target) {
                batches.push_back(b);
                b = Batch{p + 1, p + 1, 0, 0};
            }
        }
        if (b.hi > b.lo) batches.push_back(b);
        // taper the end: nothing overlaps the copy of the LAST batch, so the last batch is cut into 1/2, 1/4, 1/4
        if (batches.size() >= 2 && batches.back().cells > 400000000 && batches.back().hi - batches.back().lo >= 8) {
            const Batch last = batches.back();
            batches.pop_back();
            const double cut[2] = {0.5 * (double)last.cells, 0.75 * (double)last.cells};
            Batch t{last.lo, last.lo, 0, 0};
            int64_t acc = 0;
            int ci = 0;
            for (int64_t p = last.lo; p < last.hi; ++p) {
                t.cells += cells[p];
                t.rows += out->pair_row_base[p + 1] - out->pair_row_base[p];
                t.hi = p + 1;
                acc += cells[p];
                if (ci < 2 && (double)acc >= cut[ci]) {
                    batches.push_back(t);
                    t = Batch{p + 1, p + 1, 0, 0};
                    ++ci;
                }
            }
            if (t.hi > t.lo) batches.push_back(t);
        }
        int64_t max_pairs = 0, max_rows = 0, max_cells = 0;
        for (const Batch& q : batches) {
            max_pairs = std::max(max_pairs, q.hi - q.lo);
            max_rows = std::max(max_rows, q.rows);
            max_cells = std::max(max_cells, q.cells);
        }
        const int64_t cap = (int64_t)(beta * (double)max_cells) + 4096;
        size_t wsb = 0, worst = 0;
        int r = QP_OK;
        for (const Batch& q : batches) {
            r = qp_workspace_bytes(h_offsets, k, h_pairs + 2 * q.lo, q.hi - q.lo, &prm, cap, 0, 0, &wsb);
            if (r != QP_OK) return r;
            worst = std::max(worst, wsb);
        }
        sp = plan_slot(max_pairs, max_rows, cap, (int64_t)worst);
        if (common + 2 * sp.total <= (int64_t)workspace_bytes) break;
        if (batches.size() >= (size_t)P) {
            // one pair per batch and still too large: let qp_posteriors run with fewer scratch slots
            const int64_t spare = ((int64_t)workspace_bytes - common) / 2 - (sp.total - al256(sp.ws_bytes));
            size_t minimum = 0;
            for (const Batch& q : batches) {
                size_t mb = 0;
                const int rr = qp_workspace_bytes(h_offsets, k, h_pairs + 2 * q.lo, q.hi - q.lo, &prm, cap, 0, 1, &mb);
                if (rr != QP_ERR_WORKSPACE_TOO_SMALL && rr != QP_OK) return rr;
                minimum = std::max(minimum, mb);
            }
            if (spare < (int64_t)minimum) return QP_ERR_WORKSPACE_TOO_SMALL;
            sp = plan_slot(max_pairs, max_rows, cap, spare & ~(int64_t)255);
            break;
        }
        target *= 0.6;
        sp.total = 0;
    }
    if (sp.total == 0 || common + 2 * sp.total > (int64_t)workspace_bytes) return QP_ERR_WORKSPACE_TOO_SMALL;

    // ---- carve the device workspace ------------------------------------------------------------------------------------
    char* w = (char*)d_workspace;
    uint8_t* d_seqs = (uint8_t*)w;
    int64_t* d_offs = (int64_t*)(w + al256(seq_bytes));
    float* d_dist = (float*)(w + al256(seq_bytes) + al256((int64_t)(k + 1) * 8));
    Slot sl[2];
    cudaStream_t comp = nullptr;   // every batch's kernels, in order: two calls with their persistent kernels side by side
                                   // would starve each other's short tail kernels; a slot's own stream carries its copies
    int rc = QP_OK;
    int64_t* h_small = nullptr;   // pinned: per slot [1] nnz + [4] status
    auto cleanup = [&]() {
        for (Slot& s : sl) {
            if (s.st) cudaStreamSynchronize(s.st);
            if (s.sized) cudaEventDestroy(s.sized);
            if (s.done) cudaEventDestroy(s.done);
            if (s.st) cudaStreamDestroy(s.st);
        }
        if (comp) {
            cudaStreamSynchronize(comp);
            cudaStreamDestroy(comp);
        }
        if (h_small) cudaFreeHost(h_small);
        (void)cudaGetLastError();
    };
#define QP_H(x)                     \
    do {                            \
        if ((x) != cudaSuccess) {   \
            cleanup();              \
            return QP_ERR_CUDA;     \
        }                           \
    } while (0)
    QP_H(cudaMallocHost((void**)&h_small, 2 * 64));
    for (int q = 0; q < 16; ++q) h_small[q] = 0;
    // every copy, event and wait below goes through ck(): a failure is remembered and ends the call with QP_ERR_CUDA
    // instead of letting collect() read sizes and status words that never arrived
    bool cuda_bad = false;
    auto ck = [&](cudaError_t e) {
        if (e != cudaSuccess) cuda_bad = true;
    };
    constexpr int32_t kNotArrived = INT32_MIN;   // h_status[0] before the batch's status word has landed
    QP_H(cudaStreamCreateWithFlags(&comp, cudaStreamNonBlocking));
    for (int q = 0; q < 2; ++q) {
        Slot& s = sl[q];
        QP_H(cudaStreamCreateWithFlags(&s.st, cudaStreamNonBlocking));
        QP_H(cudaEventCreateWithFlags(&s.sized, cudaEventDisableTiming));
        QP_H(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
        char* o = w + common + q * sp.total;
        s.base = o;
        s.pairs = (int32_t*)o;
        o += al256(sp.max_pairs * 8);
        s.row_base = (int64_t*)o;
        o += al256((sp.max_pairs + 1) * 8);
        s.nnz_base = (int64_t*)o;
        o += al256((sp.max_pairs + 1) * 8);
        s.row_ptr = (int32_t*)o;
        o += al256(sp.max_rows * 4);
        s.col = (int32_t*)o;
        o += al256(sp.cap * 4);
        s.val = (float*)o;
        o += al256(sp.cap * 4);
        s.col16 = (uint16_t*)o;
        o += al256(sp.cap * 2);
        s.status = (int32_t*)o;
        o += 256;
        s.ws = o;
        s.ws_bytes = al256(sp.ws_bytes);
        s.cap = sp.cap;
        s.h_last = h_small + q * 8;
        s.h_status = (int32_t*)(h_small + q * 8 + 1);
    }

    // ---- inputs host -> device, once ---------------------------------------------------------------------------------
    cudaEvent_t up;
    QP_H(cudaEventCreateWithFlags(&up, cudaEventDisableTiming));
    ck(cudaMemcpyAsync(d_seqs, h_seqs + h_offsets[0], (size_t)seq_bytes, cudaMemcpyHostToDevice, main));
    std::vector<int64_t> shifted;   // lives until the end of the call
    if (h_offsets[0] == 0) {
        ck(cudaMemcpyAsync(d_offs, h_offsets, (size_t)(k + 1) * 8, cudaMemcpyHostToDevice, main));
    } else {   // the device copy of the sequences starts at 0; the copy is ordered on `main` like the others (earlier
               // work of the caller on that stream may still be using the workspace)
        shifted.resize(k + 1);
        for (int q = 0; q <= k; ++q) shifted[q] = h_offsets[q] - h_offsets[0];
        ck(cudaMemcpyAsync(d_offs, shifted.data(), (size_t)(k + 1) * 8, cudaMemcpyHostToDevice, main));
    }
    ck(cudaMemsetAsync(d_dist, 0, (size_t)k * k * 4, main));
    ck(cudaEventRecord(up, main));
    out->h2d_bytes += seq_bytes + (int64_t)(k + 1) * 8;
    ck(cudaStreamWaitEvent(comp, up, 0));

    // enqueue one batch: pairs up, the stage, sizes and status down -- all on the compute stream, behind the copy that
    // last read the slot's buffers
    auto enqueue = [&](Slot& s, const Batch& b) -> int {
        s.cur = b;
        const int64_t nb = b.hi - b.lo;
        s.h_status[0] = kNotArrived;   // the slot's previous batch has been collected: nothing is in flight into it
        ck(cudaStreamWaitEvent(comp, s.done, 0));
        ck(cudaMemcpyAsync(s.pairs, h_pairs + 2 * b.lo, (size_t)nb * 8, cudaMemcpyHostToDevice, comp));
        out->h2d_bytes += nb * 8;
        qp_output o;
        o.pair_row_base = s.row_base;
        o.pair_nnz_base = s.nnz_base;
        o.row_ptr = s.row_ptr;
        o.col_idx = s.col;
        o.val = s.val;
        o.nnz_capacity = s.cap;
        o.dist = d_dist;
        o.dense_P = nullptr;
        o.logZ = nullptr;
        o.status = s.status;
        const int r = qp_posteriors(d_seqs, d_offs, k, s.pairs, nb, &prm, s.ws, (size_t)s.ws_bytes, &o, comp);
        if (r != QP_OK) return r;
        if (out->col_idx16) k_narrow_cols<<<1184, 256, 0, comp>>>(s.col, s.nnz_base + nb, s.cap, s.col16);
        ck(cudaMemcpyAsync(s.h_last, s.nnz_base + nb, 8, cudaMemcpyDeviceToHost, comp));
        ck(cudaMemcpyAsync(s.h_status, s.status, 16, cudaMemcpyDeviceToHost, comp));
        ck(cudaEventRecord(s.sized, comp));
        // what does not depend on the CSR size goes down on the slot's copy stream right away
        ck(cudaStreamWaitEvent(s.st, s.sized, 0));
        ck(cudaMemcpyAsync(out->row_ptr + out->pair_row_base[b.lo], s.row_ptr, (size_t)b.rows * 4, cudaMemcpyDeviceToHost, s.st));
        ck(cudaMemcpyAsync(out->pair_nnz_base + b.lo + 1, s.nnz_base + 1, (size_t)nb * 8, cudaMemcpyDeviceToHost, s.st));
        out->d2h_bytes += 24 + b.rows * 4 + nb * 8;
        return cudaGetLastError() == cudaSuccess && !cuda_bad ? QP_OK : QP_ERR_CUDA;
    };

    // ---- the pipeline ---------------------------------------------------------------------------------------------------
    // work list: batches in order; a batch whose CSR does not fit its slot is split in two and taken again
    std::vector<Batch> work(batches.rbegin(), batches.rend());   // stack: next batch at the back
    int64_t nnz_running = 0;     // entries of the batches collected so far
    int64_t required = 0;        // entries needed in all (keeps counting past the caller's capacity)
    bool host_overflow = false;
    std::vector<int> inflight;   // slots in enqueue order
    int next_slot = 0;
    struct Fixup {
        int64_t lo, hi, base;
        int slot;
    };
    std::vector<Fixup> fixups;   // pair_nnz_base ranges waiting for their copy to land
    auto apply_fixups = [&](int slot) {   // after the slot's `done` event has completed
        for (size_t u = 0; u < fixups.size();) {
            if (fixups[u].slot != slot) {
                ++u;
                continue;
            }
            for (int64_t p = fixups[u].lo + 1; p <= fixups[u].hi; ++p) out->pair_nnz_base[p] += fixups[u].base;
            fixups.erase(fixups.begin() + u);
        }
    };
    auto collect = [&](int q) -> int {   // sizes known -> CSR down -> fix the prefix; returns QP_OK, an error, or 1 = "split"
        Slot& s = sl[q];
        if (cudaEventSynchronize(s.sized) != cudaSuccess || cuda_bad) return QP_ERR_CUDA;
        const int code = s.h_status[0];
        if (code == kNotArrived) return QP_ERR_CUDA;   // the status word of this batch never landed
        const Batch b = s.cur;
        const int64_t nb = b.hi - b.lo;
        if (code == QP_ERR_NNZ_CAPACITY && nb > 1) return 1;
        if (code != QP_OK) {
            out->status[0] = code;
            out->status[1] = s.h_status[1] >= 0 ? (int32_t)(b.lo + s.h_status[1]) : -1;
            return code;
        }
        const int64_t nz = *s.h_last;
        out->status[3] += s.h_status[3];
        required += nz;
        if (nnz_running + nz > out->nnz_capacity) {
            host_overflow = true;
        } else {
            if (out->col_idx16) ck(cudaMemcpyAsync(out->col_idx16 + nnz_running, s.col16, (size_t)nz * 2, cudaMemcpyDeviceToHost, s.st));
            else ck(cudaMemcpyAsync(out->col_idx + nnz_running, s.col, (size_t)nz * 4, cudaMemcpyDeviceToHost, s.st));
            ck(cudaMemcpyAsync(out->val + nnz_running, s.val, (size_t)nz * 4, cudaMemcpyDeviceToHost, s.st));
            out->d2h_bytes += nz * (out->col_idx16 ? 6 : 8);
        }
        ck(cudaEventRecord(s.done, s.st));
        if (cuda_bad) return QP_ERR_CUDA;
        s.out_nnz0 = nnz_running;   // the batch's pair_nnz_base arrives as local offsets: made global once `done` has passed
        nnz_running += nz;
        ++out->batches;
        fixups.push_back({b.lo, b.hi, s.out_nnz0, q});
        return QP_OK;
    };
    while (rc == QP_OK && (!work.empty() || !inflight.empty())) {
        // keep two batches in flight
        while (rc == QP_OK && !work.empty() && inflight.size() < 2) {
            Slot& s = sl[next_slot];   // (its kernels wait on the device for the slot's previous copy: enqueue)
            rc = enqueue(s, work.back());
            work.pop_back();
            inflight.push_back(next_slot);
            next_slot ^= 1;
        }
        if (rc != QP_OK) break;
        const int q = inflight.front();
        const int r = collect(q);
        if (r == 1) {
            // denser than beta_guess: everything enqueued after this batch is abandoned (its results are simply
            // computed again), the batch goes back as two halves
            ck(cudaStreamSynchronize(comp));
            for (int other : inflight) ck(cudaStreamSynchronize(sl[other].st));
            for (size_t u = inflight.size(); u-- > 1;) work.push_back(sl[inflight[u]].cur);
            const Batch b = sl[q].cur;
            int64_t mid = b.lo, acc = 0;
            while (mid < b.hi - 1 && acc + cells[mid] <= b.cells / 2) acc += cells[mid++];
            if (mid == b.lo) mid = b.lo + 1;
            Batch hi_half{mid, b.hi, 0, 0}, lo_half{b.lo, mid, 0, 0};
            for (int64_t p = b.lo; p < b.hi; ++p) {
                Batch& t = p < mid ? lo_half : hi_half;
                t.cells += cells[p];
                t.rows += out->pair_row_base[p + 1] - out->pair_row_base[p];
            }
            work.push_back(hi_half);
            work.push_back(lo_half);
            inflight.clear();
            next_slot = 0;
            ck(cudaEventRecord(sl[0].done, sl[0].st));
            ck(cudaEventRecord(sl[1].done, sl[1].st));
            if (cuda_bad) rc = QP_ERR_CUDA;
            continue;
        }
        rc = r;
        inflight.erase(inflight.begin());
    }
    ck(cudaStreamSynchronize(comp));
    for (int q = 0; q < 2; ++q) {
        ck(cudaStreamSynchronize(sl[q].st));
        if (rc == QP_OK && cuda_bad) rc = QP_ERR_CUDA;
        if (rc == QP_OK) apply_fixups(q);
    }
    if (rc == QP_OK) {
        ck(cudaMemcpyAsync(out->dist, d_dist, (size_t)k * k * 4, cudaMemcpyDeviceToHost, main));
        out->d2h_bytes += (int64_t)k * k * 4;
        if (cudaStreamSynchronize(main) != cudaSuccess || cuda_bad) rc = QP_ERR_CUDA;
    }
    cudaEventDestroy(up);
    cleanup();
#undef QP_H
    if (rc == QP_OK && host_overflow) {
        rc = QP_ERR_NNZ_CAPACITY;
        out->pair_nnz_base[P] = required;
    }
    if (rc != QP_OK && out->status[0] == 0) out->status[0] = rc;
    return rc;
}
