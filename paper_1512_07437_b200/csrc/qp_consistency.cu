// qp_consistency.cu -- stage III: selective consistency transformation of the sparse posterior matrices
// (include/qp.h qp_consistency).
//
// "consistency relies on the relaxation of posterior probability matrices by other sequences";
// PAPER.md:55 / :63 (Figure 2): S_xy is relaxed over z iff f(d_xz, d_yz) <= T on the tree-guided distance;
// PAPER.md:57 / :65 / :109: the original signal is amplified by h_xy in [1, h]; PAPER.md:59 (footnote): sparse form.
// The formula (the paper prints none):
//     S'_xy = ( 2 h_xy S_xy + sum_{z in sel(x,y)} S_xz S_zy ) / ( 2 h_xy + |sel(x,y)| )   on the pattern of S_xy,
//     h_xy = 1 + (h - 1) min(|sel|, R) / R,   values below tau dropped.
//
// Design (measured: INSTRUCTION-bound, not bandwidth-bound -- ~350 warp instructions per (row, z) for ~4.5 useful
// multiply-adds at 15 of 32 lanes, DRAM at 2 % of peak, profiles/r02_stage3.md; the algorithmic ratio is ~1 multiply-add
// per 5 bytes read):
//   k_cs_index      pair lookup table pair_of[k][k] -> (pair, orientation); per-pair column counts
//   k_cs_transpose  per pair: an interleaved (value, column) copy of the matrix and its transpose (value, row), so
//                   that EVERY oriented matrix S_ab (rows = residues of a) is a row-compressed list of 8-byte entries
//   k_cs_relax      one CTA per pair; for every selected z (outer loop) the warps take the rows i of S_xy, lane q owns
//                   the q-th stored cell (i, c_q) of the row:
//                   S_xz S_zy (i, c_q) = sum_k S_xz(i,k) S_yz(c_q,k) = <row i of S_xz , row c_q of S_yz>. The warp
//                   spreads row i of S_xz into a dense window over k in shared memory; every lane walks its own row
//                   of S_yz and gathers from the window: no atomics, no search, a fixed summation order (z ascending,
//                   k ascending), so the result is reproducible bit for bit. With z outermost the two factor
//                   matrices stream through L1 once per (pair, z); the accumulators sit in shared memory.
//   k_scan / k_cs_place   kept entries -> the caller's CSR in pair order.
#include <cuda_runtime.h>

#include <cstdint>

#include "qp.h"
#include "qp_scan.cuh"

namespace qp {

constexpr int kCsThreads = 256;
constexpr int kCsWarps = kCsThreads / 32;
constexpr int kCsWin = 128;          // generic routine: dense window over k (floats per warp)
constexpr int kCsList = kCsThreads;  // selected sequences held in shared memory at a time: one block of candidates
constexpr int kCsAcc = 8192;         // accumulators (cells of S_xy) held in shared memory; larger pairs use the staging area
constexpr unsigned kAll = 0xffffffffu;

struct CsHeader {
    int32_t status[4];
};

struct CsZ {                 // one selected sequence z, both factors as row-compressed lists
    const int32_t* rpA;      // row pointer of S_xz (rows = residues of x), local offsets
    const float2* entA;      // its entries (value, k)
    const int32_t* rpB;      // row pointer of S_yz (rows = residues of y)
    const float2* entB;
};

struct CsArgs {
    const int64_t* offs;
    const int32_t* pairs;
    int64_t P;
    int32_t k;
    // input CSR (layout of qp_output)
    const int64_t* row_base;
    const int64_t* nnz_base;
    const int32_t* row_ptr;
    const int32_t* col_idx;
    const float* val;
    const int32_t* treedist;
    int32_t T, f, max_relax;
    float h, tau;
    // workspace
    CsHeader* hdr;
    int32_t* pair_of;        // [k][k]: 2 * pair + (1 if the pair is stored the other way round), -1 if absent
    int32_t* cols1;          // [P] m_p + 1
    int64_t* col_base;       // [P+1] prefix of cols1
    int64_t rpT_cap;         // ints available for rpT / curT
    float2* ent;             // [2][nnz]: direct (value, column) and transposed (value, row) entries
    int64_t nnz;
    int32_t* rpT;            // [sum(m_p+1)] row pointer of the transposed matrices
    int32_t* curT;           // [sum(m_p+1)] scatter cursors
    float2* tmp;             // [nnz] partial sums, then the kept (value, column) entries at their input row start
    int32_t* nnz_pair;       // [P]
    // output
    int64_t* out_nnz_base;
    int32_t* out_row_ptr;
    int32_t* out_col;
    float* out_val;
    int64_t out_cap;
    int32_t* relaxations;
};

__device__ __forceinline__ void cs_status(CsHeader* h, int code, int where) {
    if (atomicCAS(&h->status[0], 0, code) == 0) h->status[1] = where;
}

__global__ void k_cs_index(CsArgs a) {
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= a.P) return;
    const int x = a.pairs[2 * p], y = a.pairs[2 * p + 1];
    int32_t c1 = 1;
    if (x < 0 || y < 0 || x >= a.k || y >= a.k || x == y) {
        cs_status(a.hdr, QP_ERR_BAD_PAIR, (int)p);
    } else {
        const int64_t n = a.offs[x + 1] - a.offs[x], m = a.offs[y + 1] - a.offs[y];
        if (n < 1 || m < 1 || n > QP_MAX_LEN || m > QP_MAX_LEN) {
            cs_status(a.hdr, QP_ERR_EMPTY_SEQUENCE, (int)p);
        } else {
            a.pair_of[(int64_t)x * a.k + y] = (int32_t)(2 * p);
            a.pair_of[(int64_t)y * a.k + x] = (int32_t)(2 * p + 1);
            c1 = (int32_t)m + 1;
        }
    }
    a.cols1[p] = c1;
}

// in-place exclusive prefix over v[0..len) by the whole block; v[len] is NOT touched. Returns the total.
__device__ int block_scan_inplace(int32_t* v, int len, int32_t* sh /*[kCsThreads]*/) {
    const int t = threadIdx.x, per = (len + kCsThreads - 1) / kCsThreads;
    const int lo = min(len, t * per), hi = min(len, (t + 1) * per);
    int s = 0;
    for (int q = lo; q < hi; ++q) s += v[q];
    sh[t] = s;
    __syncthreads();
    for (int o = 1; o < kCsThreads; o <<= 1) {
        const int u = t >= o ? sh[t - o] : 0;
        __syncthreads();
        sh[t] += u;
        __syncthreads();
    }
    int run = sh[t] - s;
    const int total = sh[kCsThreads - 1];
    for (int q = lo; q < hi; ++q) {
        const int c = v[q];
        v[q] = run;
        run += c;
    }
    __syncthreads();
    return total;
}

__global__ void __launch_bounds__(kCsThreads) k_cs_transpose(CsArgs a) {
    __shared__ int32_t sh[kCsThreads];
    const int64_t p = blockIdx.x;
    const int x = a.pairs[2 * p], y = a.pairs[2 * p + 1];
    if (a.hdr->status[0] != 0) return;
    const int n = (int)(a.offs[x + 1] - a.offs[x]), m = (int)(a.offs[y + 1] - a.offs[y]);
    if (a.col_base[a.P] > a.rpT_cap) {
        if (p == 0 && threadIdx.x == 0) cs_status(a.hdr, QP_ERR_WORKSPACE_TOO_SMALL, -1);
        return;
    }
    // S_xz is a factor of some relaxation only if f(d_xz, .) <= T is possible: for max and sum that needs d_xz <= T
    // (distances are >= 0). Copies of the other pairs are never read.
    const int32_t* rp = a.row_ptr + a.row_base[p];
    const int64_t base = a.nnz_base[p];
    const int cnt = rp[n];
    if (base + cnt > a.nnz) {   // checked for EVERY pair, copied or not: the later kernels index tmp / ent with base + e
        if (threadIdx.x == 0) cs_status(a.hdr, QP_ERR_NNZ_CAPACITY, (int)p);
        return;
    }
    if (a.f != QP_SEL_MIN && a.treedist[(int64_t)x * a.k + y] > a.T) return;
    const int32_t* col = a.col_idx + base;
    const float* val = a.val + base;
    float2* e0 = a.ent + base;             // direct, interleaved
    float2* e1 = a.ent + a.nnz + base;     // transposed
    int32_t* rT = a.rpT + a.col_base[p];   // m + 1 entries
    int32_t* cur = a.curT + a.col_base[p];
    for (int j = threadIdx.x; j <= m; j += kCsThreads) rT[j] = 0;
    __syncthreads();
    for (int e = threadIdx.x; e < cnt; e += kCsThreads) {
        const int j = col[e];
        e0[e] = make_float2(val[e], __int_as_float(j));
        atomicAdd(&rT[j], 1);                      // count of column j (shifted into place by the exclusive scan)
    }
    __syncthreads();
    block_scan_inplace(rT, m, sh);                 // rT[j] = entries in columns < j
    if (threadIdx.x == 0) rT[m] = cnt;
    for (int j = threadIdx.x; j < m; j += kCsThreads) cur[j] = rT[j];
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += kCsThreads)
        for (int e = rp[i]; e < rp[i + 1]; ++e) {
            const int pos = atomicAdd(&cur[col[e]], 1);
            e1[pos] = make_float2(val[e], __int_as_float(i));
        }
    __syncthreads();
    // rows of a column arrive in any order: sort every column's (short) segment by row
    for (int j = threadIdx.x; j < m; j += kCsThreads) {
        const int lo = rT[j], hi = j + 1 < m ? rT[j + 1] : cnt;
        for (int u = lo + 1; u < hi; ++u) {
            const float2 key = e1[u];
            int v = u - 1;
            while (v >= lo && __float_as_int(e1[v].y) > __float_as_int(key.y)) {
                e1[v + 1] = e1[v];
                --v;
            }
            e1[v + 1] = key;
        }
    }
}

// oriented matrix S_ab (rows = residues of a): row pointer and entry list, from the pair table
__device__ __forceinline__ bool cs_oriented(const CsArgs& a, int ra, int rb, const int32_t*& rp, const float2*& ent) {
    const int code = a.pair_of[(int64_t)ra * a.k + rb];
    if (code < 0) return false;
    const int64_t p = code >> 1;
    if (code & 1) {
        rp = a.rpT + a.col_base[p];
        ent = a.ent + a.nnz + a.nnz_base[p];
    } else {
        rp = a.row_ptr + a.row_base[p];
        ent = a.ent + a.nnz_base[p];
    }
    return true;
}

// ---- the inner routine of the relaxation ----------------------------------------------------------------------------
// Adds, for one selected z, <row i of S_xz, row c of S_yz> to the accumulator of the stored cells (i, c) of row i of
// S_xy, cells [lo, hi), 32 at a time (one per lane). Any row lengths, any spread of k: row i of S_xz is spread into a
// dense window over k in shared memory, kCsWin wide, as many windows as its spread needs (normally one); every lane
// walks its own row of S_yz and gathers from the window. `w` is the warp's window, all zero between uses.
template <typename AccT>
__device__ __forceinline__ void cs_row_generic(const CsZ& Z, int i, int lo, int hi, const int32_t* __restrict__ colxy,
                                               AccT accum, float* w, int lane) {
    const int a0 = Z.rpA[i], a1 = Z.rpA[i + 1];
    if (a0 == a1) return;                                  // warp-uniform: x_i has no partner in z
    for (int qb = lo; qb < hi; qb += 32) {
        const int e = qb + lane;
        const bool have = e < hi;
        int b0 = 0, b1 = 0;
        if (have) {
            const int cq = __ldg(colxy + e);
            b0 = Z.rpB[cq];
            b1 = Z.rpB[cq + 1];
        }
        float accv = 0.f;
        for (int ab = a0; ab < a1; ab += 32) {             // row i of S_xz, 32 entries at a time
            const bool ha = ab + lane < a1;
            float av = 0.f;
            int ak = 0;
            if (ha) {
                const float2 t = __ldg(Z.entA + ab + lane);
                av = t.x;
                ak = __float_as_int(t.y);
            }
            const int na = min(32, a1 - ab);
            const int kmin = __shfl_sync(kAll, ak, 0), kmax = __shfl_sync(kAll, ak, na - 1);
            for (int wb = kmin; wb <= kmax; wb += kCsWin) {   // dense window over k (normally one)
                const bool inw = ha && (unsigned)(ak - wb) < (unsigned)kCsWin;
                if (inw) w[ak - wb] = av;
                __syncwarp();
                // row c_q of S_yz against the window, four entries per round of loads; entries outside the window
                // meet zeros or fail the range test
                for (int b = b0; b < b1; b += 4) {
                    float2 t[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        t[u] = b + u < b1 ? __ldg(Z.entB + b + u) : make_float2(0.f, __int_as_float(-(1 << 30)));
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int d = __float_as_int(t[u].y) - wb;
                        if ((unsigned)d < (unsigned)kCsWin) accv = fmaf(w[d], t[u].x, accv);
                    }
                }
                __syncwarp();
                if (inw) w[ak - wb] = 0.f;
            }
        }
        if (have) accum(e, accv);
    }
}

// One CTA per pair (x, y). The selected sequences are taken a block of candidates at a time, in ascending order; for
// every selected z (outer loop, the whole CTA on the same z so that its two matrices stream through L1 once) the
// warps take the rows of S_xy (inner loop) and add <row i of S_xz, row c of S_yz> to the accumulator of every stored
// cell (i, c). Pairs with at most kCsAcc cells keep the accumulators in shared memory, larger ones in the staging area.
__global__ void __launch_bounds__(kCsThreads) k_cs_relax(CsArgs a) {
    __shared__ CsZ zl[kCsList];
    __shared__ float win[kCsWarps][kCsWin];
    __shared__ float acc_s[kCsAcc];                                  // accumulators of S_xy's stored cells
    __shared__ int32_t sh[kCsThreads];
    __shared__ int wcnt[kCsWarps];
    __shared__ int rtot;
    const int64_t p = blockIdx.x;
    if (a.hdr->status[0] != 0) return;
    const int x = a.pairs[2 * p], y = a.pairs[2 * p + 1];
    const int n = (int)(a.offs[x + 1] - a.offs[x]);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t* __restrict__ rp = a.row_ptr + a.row_base[p];
    const int64_t base = a.nnz_base[p];
    const int cnt = rp[n];
    const int32_t* __restrict__ colxy = a.col_idx + base;
    const float* __restrict__ valxy = a.val + base;
    float2* tmp = a.tmp + base;
    int32_t* orp = a.out_row_ptr + a.row_base[p];
    const int32_t* tdx = a.treedist + (int64_t)x * a.k;
    const int32_t* tdy = a.treedist + (int64_t)y * a.k;
    const bool cached = cnt <= kCsAcc;                   // CTA-uniform: the accumulators live in shared memory
    float* w = win[warp];
    for (int u = lane; u < kCsWin; u += 32) w[u] = 0.f;   // the window is all zero between uses
    if (tid == 0) rtot = 0;
    __syncthreads();
    bool touched = false;
    for (int z0 = 0; z0 < a.k; z0 += kCsThreads) {
        // ---- selection: candidates z0 .. z0+255, listed in ascending order ---------------------------
        const int z = z0 + tid;
        CsZ mine;
        bool sel = false;
        if (z < a.k && z != x && z != y) {
            const int dx = tdx[z], dy = tdy[z];
            const int fv = a.f == QP_SEL_MAX ? max(dx, dy) : (a.f == QP_SEL_MIN ? min(dx, dy) : dx + dy);
            if (fv <= a.T) sel = cs_oriented(a, x, z, mine.rpA, mine.entA) && cs_oriented(a, y, z, mine.rpB, mine.entB);
        }
        const unsigned bal = __ballot_sync(kAll, sel);
        if (lane == 0) wcnt[warp] = __popc(bal);
        __syncthreads();
        int off = 0, nz = 0;
        for (int q = 0; q < kCsWarps; ++q) {
            if (q < warp) off += wcnt[q];
            nz += wcnt[q];
        }
        if (sel) zl[off + __popc(bal & ((1u << lane) - 1))] = mine;
        if (tid == 0) rtot += nz;
        if (nz > 0 && !touched) {   // CTA-uniform: the first selected sequences of this pair
            if (cached) for (int e = tid; e < cnt; e += kCsThreads) acc_s[e] = 0.f;
            else for (int e = tid; e < cnt; e += kCsThreads) tmp[e].x = 0.f;
            touched = true;
        }
        __syncthreads();
        // ---- relax over the listed sequences ------------------------------------------------------------------------
        for (int q = 0; q < nz; ++q) {
            const CsZ Z = zl[q];
            if (cached) {
                auto add_s = [&](int e, float v) { acc_s[e] += v; };
                for (int i = warp; i < n; i += kCsWarps) cs_row_generic(Z, i, rp[i], rp[i + 1], colxy, add_s, w, lane);
            } else {
                auto add_g = [&](int e, float v) { tmp[e].x += v; };
                for (int i = warp; i < n; i += kCsWarps) cs_row_generic(Z, i, rp[i], rp[i + 1], colxy, add_g, w, lane);
            }
        }
        __syncthreads();   // the list is rebuilt by the next block of candidates
    }
    // ---- amplify, normalise, threshold; kept entries are packed at the start of their row ------------
    const int r = rtot;
    if (!touched) {   // nothing selected: S' = S cut at the threshold
        // a stage-III threshold above the one the input was cut at drops entries here too (include/qp.h: "values below
        // `threshold` are dropped", whatever |sel| is); only when every entry passes -- the usual case, the same tau in
        // both stages -- does the placement copy the input entries themselves
        int below = 0;
        for (int e = tid; e < cnt; e += kCsThreads) below |= valxy[e] < a.tau;
        below = __syncthreads_or(below);
        if (below) {   // CTA-uniform: zero accumulators, then the general path with r = 0 gives v = (2 S + 0) / 2 = S exactly
            if (cached) for (int e = tid; e < cnt; e += kCsThreads) acc_s[e] = 0.f;
            else for (int e = tid; e < cnt; e += kCsThreads) tmp[e].x = 0.f;
            touched = true;
            __syncthreads();
        }
    }
    if (!touched) {
        for (int i = tid; i <= n; i += kCsThreads) orp[i] = rp[i];
        if (tid == 0) {
            a.nnz_pair[p] = -cnt - 1;                          // negative: "copy from the input"
            if (a.relaxations) a.relaxations[p] = 0;
        }
        return;
    }
    const float hxy = 1.f + (a.h - 1.f) * (float)min(r, a.max_relax) / (float)a.max_relax;
    const float w2 = 2.f * hxy, inv = 1.f / (w2 + (float)r);
    for (int i = warp; i < n; i += kCsWarps) {
        const int s0 = rp[i], s1 = rp[i + 1];
        int kept = 0;
        for (int qb = s0; qb < s1; qb += 32) {
            const int e = qb + lane;
            const bool have = e < s1;
            float v = 0.f;
            int cq = 0;
            if (have) {
                cq = colxy[e];
                v = fmaf(w2, valxy[e], cached ? acc_s[e] : tmp[e].x) * inv;
            }
            const bool keep = have && v >= a.tau;
            const unsigned kb = __ballot_sync(kAll, keep);
            if (keep) tmp[s0 + kept + __popc(kb & ((1u << lane) - 1))] = make_float2(v, __int_as_float(cq));
            kept += __popc(kb);
        }
        if (lane == 0) orp[i] = kept;
    }
    __syncthreads();
    // ---- row counts -> row pointer of the relaxed pair ---------------------------------------------------------------
    const int total = block_scan_inplace(orp, n, sh);
    if (tid == 0) {
        orp[n] = total;
        a.nnz_pair[p] = total;
        if (a.relaxations) a.relaxations[p] = r;
    }
}

// nnz_pair holds -(count) - 1 for the pairs that were not relaxed: make it the count and keep the sign as a flag
// for the placement
__global__ void k_cs_counts(CsArgs a, int32_t* flags) {
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= a.P) return;
    const int v = a.nnz_pair[p];
    flags[p] = v < 0;
    if (v < 0) a.nnz_pair[p] = -v - 1;
}

__global__ void __launch_bounds__(kCsThreads) k_cs_place(CsArgs a, const int32_t* __restrict__ flags) {
    const int64_t p = blockIdx.x;
    if (a.hdr->status[0] != 0) return;
    const int x = a.pairs[2 * p];
    const int n = (int)(a.offs[x + 1] - a.offs[x]);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t* rp = a.row_ptr + a.row_base[p];
    const int32_t* orp = a.out_row_ptr + a.row_base[p];
    const int64_t ib = a.nnz_base[p], ob = a.out_nnz_base[p];
    if (ob + orp[n] > a.out_cap) {
        if (threadIdx.x == 0) cs_status(a.hdr, QP_ERR_NNZ_CAPACITY, (int)p);
        return;
    }
    if (flags[p]) {   // not relaxed: the input entries, unchanged
        const int c = orp[n];
        for (int e = threadIdx.x; e < c; e += kCsThreads) {
            a.out_val[ob + e] = a.val[ib + e];
            a.out_col[ob + e] = a.col_idx[ib + e];
        }
        return;
    }
    const float2* tmp = a.tmp + ib;
    for (int i = warp; i < n; i += kCsWarps) {
        const int s0 = rp[i], d0 = orp[i], c = orp[i + 1] - d0;
        for (int q = lane; q < c; q += 32) {
            const float2 t = tmp[s0 + q];
            a.out_val[ob + d0 + q] = t.x;
            a.out_col[ob + d0 + q] = __float_as_int(t.y);
        }
    }
}

__global__ void k_cs_finish(const CsHeader* h, int32_t* status) {
    if (threadIdx.x < 4) status[threadIdx.x] = h->status[threadIdx.x];
}

static inline int64_t al256(int64_t v) { return (v + 255) & ~(int64_t)255; }

struct CsLayout {
    int64_t hdr, pair_of, cols1, col_base, ent, tmp, nnz_pair, flags, rpT, curT, total;
};
static CsLayout cs_layout(int32_t k, int64_t P, int64_t nnz, int64_t cols_total) {
    CsLayout L;
    int64_t o = 0;
    auto take = [&](int64_t b) {
        const int64_t r = o;
        o += al256(b);
        return r;
    };
    L.hdr = take(sizeof(CsHeader));
    L.pair_of = take((int64_t)k * k * 4);
    L.cols1 = take(P * 4);
    L.col_base = take((P + 1) * 8);
    L.ent = take(2 * nnz * 8);
    L.tmp = take(nnz * 8);
    L.nnz_pair = take(P * 4);
    L.flags = take(P * 4);
    L.rpT = take(cols_total * 4);     // the two arrays sized by sum(m_p + 1) come last: the device checks the sum
    L.curT = take(cols_total * 4);
    L.total = o;
    return L;
}

}  // namespace qp

using namespace qp;

extern "C" int qp_consistency_passes(int32_t k) { return k < 50 ? 2 : 1; }

extern "C" int qp_consistency_workspace_bytes(const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P,
                                              int64_t nnz, size_t* out_bytes) {
    if (!h_offsets || (!h_pairs && P > 0) || !out_bytes || k < 0 || P < 0 || nnz < 0) return QP_ERR_INVALID_ARG;
    int64_t cols = 0;
    for (int64_t p = 0; p < P; ++p) {
        const int x = h_pairs[2 * p], y = h_pairs[2 * p + 1];
        if (x < 0 || y < 0 || x >= k || y >= k || x == y) return QP_ERR_BAD_PAIR;
        const int64_t m = h_offsets[y + 1] - h_offsets[y];
        if (m < 1 || m > QP_MAX_LEN) return QP_ERR_EMPTY_SEQUENCE;
        cols += m + 1;
    }
    *out_bytes = (size_t)cs_layout(k, P, nnz, cols).total;
    return QP_OK;
}

extern "C" int qp_consistency(const int64_t* d_offsets, int32_t k, const int32_t* d_pairs, int64_t P, const qp_csr* in,
                              int64_t nnz, const int32_t* d_treedist, const qp_consistency_params* prm,
                              void* d_workspace, size_t workspace_bytes, const qp_csr_out* out, void* cuda_stream) {
    if (!in || !out || !prm || k < 0 || P < 0 || P > 0x7fffffff || nnz < 0) return QP_ERR_INVALID_ARG;
    if (!out->pair_nnz_base || !out->status) return QP_ERR_INVALID_ARG;
    if (!(prm->h >= 1.0) || prm->max_relax < 1 || !(prm->threshold >= 0.0) || prm->f < QP_SEL_MAX || prm->f > QP_SEL_SUM)
        return QP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (P == 0) {
        if (cudaMemsetAsync(out->pair_nnz_base, 0, 8, st) != cudaSuccess || cudaMemsetAsync(out->status, 0, 16, st) != cudaSuccess)
            return QP_ERR_CUDA;
        return QP_OK;
    }
    if (!d_offsets || !d_pairs || !d_treedist || !d_workspace || !in->pair_row_base || !in->pair_nnz_base || !in->row_ptr ||
        !out->row_ptr)
        return QP_ERR_INVALID_ARG;
    if (nnz > 0 && (!in->col_idx || !in->val || !out->col_idx || !out->val)) return QP_ERR_INVALID_ARG;
    if (out->nnz_capacity < 0 || ((uintptr_t)d_workspace & 255) != 0) return QP_ERR_INVALID_ARG;
    // everything but the two arrays sized by sum(m_p + 1) has a host-known size; what is left goes to those two
    const CsLayout L = cs_layout(k, P, nnz, 0);
    if ((int64_t)workspace_bytes < L.total + 512) return QP_ERR_WORKSPACE_TOO_SMALL;
    const int64_t tail_ints = (((int64_t)workspace_bytes - L.rpT) / 2 / 256) * 256 / 4;
    char* ws = (char*)d_workspace;
    CsArgs a;
    a.offs = d_offsets;
    a.pairs = d_pairs;
    a.P = P;
    a.k = k;
    a.row_base = in->pair_row_base;
    a.nnz_base = in->pair_nnz_base;
    a.row_ptr = in->row_ptr;
    a.col_idx = in->col_idx;
    a.val = in->val;
    a.treedist = d_treedist;
    a.T = prm->T;
    a.f = prm->f;
    a.max_relax = prm->max_relax;
    a.h = (float)prm->h;
    a.tau = (float)prm->threshold;
    a.hdr = (CsHeader*)(ws + L.hdr);
    a.pair_of = (int32_t*)(ws + L.pair_of);
    a.cols1 = (int32_t*)(ws + L.cols1);
    a.col_base = (int64_t*)(ws + L.col_base);
    a.rpT_cap = tail_ints;
    a.ent = (float2*)(ws + L.ent);
    a.nnz = nnz;
    a.rpT = (int32_t*)(ws + L.rpT);
    a.curT = a.rpT + tail_ints;
    a.tmp = (float2*)(ws + L.tmp);
    a.nnz_pair = (int32_t*)(ws + L.nnz_pair);
    a.out_nnz_base = out->pair_nnz_base;
    a.out_row_ptr = out->row_ptr;
    a.out_col = out->col_idx;
    a.out_val = out->val;
    a.out_cap = out->nnz_capacity;
    a.relaxations = out->relaxations;
#define QP_CS(x)                                    \
    do {                                            \
        if ((x) != cudaSuccess) return QP_ERR_CUDA; \
    } while (0)
    QP_CS(cudaMemsetAsync(a.hdr, 0, sizeof(CsHeader), st));
    QP_CS(cudaMemsetAsync(a.pair_of, 0xff, (size_t)k * k * 4, st));
    k_cs_index<<<(int)((P + 255) / 256), 256, 0, st>>>(a);
    k_scan<int32_t><<<1, 1024, 0, st>>>(a.cols1, P, a.col_base);
    k_cs_transpose<<<(int)P, kCsThreads, 0, st>>>(a);
    k_cs_relax<<<(int)P, kCsThreads, 0, st>>>(a);
    int32_t* flags = (int32_t*)(ws + L.flags);
    k_cs_counts<<<(int)((P + 255) / 256), 256, 0, st>>>(a, flags);
    k_scan<int32_t><<<1, 1024, 0, st>>>(a.nnz_pair, P, a.out_nnz_base);
    k_cs_place<<<(int)P, kCsThreads, 0, st>>>(a, flags);
    k_cs_finish<<<1, 32, 0, st>>>(a.hdr, out->status);
    QP_CS(cudaGetLastError());
#undef QP_CS
    return QP_OK;
}
