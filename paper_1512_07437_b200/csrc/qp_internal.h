// qp_internal.h -- data layout shared by the scheduler kernels, the pair kernels and the host API.
#pragma once
#include <stdint.h>

#include "qp_lane.h"
#include "qp_both.cuh"

namespace qp {

#if defined(__CUDACC__)
#define QP_HD2 __host__ __device__ constexpr inline
#else
#define QP_HD2 constexpr inline
#endif

// Scheduling classes. A class fixes the stripe width C (columns per lane) and the number W of warps that share one
// pair. W = 1 ("packed"): every warp of a CTA works on a pair of its own, the pair's columns fit one 32*C-column
// block. W > 1 ("split"): the W warps of a CTA take W neighbouring column blocks of ONE pair and run them as a
// pipelined anti-diagonal wavefront, block boundaries handed over through shared memory (qp_pair.cuh).
//   class 0..14  : packed, C = c + 2 = 2..16                (fp64: only C = 2, 4, 6, 8 exist)
//   class 15..17 : split,  fp32 (C, W) = (8,4) (12,4) (16,4);  fp64 (C, W) = (2,8) (4,8) (8,8)
//   class 18..21 : packed TWO-BLOCK, fp32 only, C = c - 18 + 9 = 9..12: a pair of 513..768 columns and moderate size
//                  on ONE warp, which runs its two 32*C-column blocks one after the other (the boundary column goes
//                  through the scratch slot). Separate kernel instances (MODE | kModeMB): a run-time block count in
//                  the one-block kernels costs them registers they do not have (measured: 5-9 % slower).
constexpr int kNumClasses = 22;
constexpr int kNumPacked = 15;        // classes below: packed one-block
constexpr int kSplitEnd = 18;         // classes kNumPacked .. kSplitEnd-1: split; from kSplitEnd on: packed two-block
constexpr int kModeMB = 4;            // MODE bit of the two-block instances (qp_pair.cuh)
constexpr int kWarpsPerCta = 4;       // packed classes
constexpr int kNumBins = 384;         // size bins: 8 per octave of scratch bytes
constexpr int kSmAssumed = 148;       // used by the host-only workspace query when no device is visible

QP_HD2 int class_C(int c, bool fp64) {
    if (c < kNumPacked) return (fp64 && (c > 6 || (c & 1))) ? 0 : c + 2;
    if (c >= kSplitEnd) return fp64 ? 0 : c - kSplitEnd + 9;
    return fp64 ? (c == 15 ? 2 : (c == 16 ? 4 : 8)) : (c == 15 ? 8 : (c == 16 ? 12 : 16));
}
QP_HD2 int class_W(int c, bool fp64) { return (c < kNumPacked || c >= kSplitEnd) ? 1 : (fp64 ? 8 : 4); }
QP_HD2 int class_index(int C, int W, bool fp64, bool two_block) {
    if (two_block) return kSplitEnd + C - 9;
    if (W == 1) return C - 2;
    return fp64 ? (C == 2 ? 15 : (C == 4 ? 16 : 17)) : (C == 8 ? 15 : (C == 12 ? 16 : 17));
}
constexpr uint32_t kMaskF32 = 0x3fffff;    // fp32 pass: packed C = 2..16, the three split classes, two-block C = 9..12
constexpr uint32_t kMaskF64 = 0x20055;     // QP_FP64: packed C = 2, 4, 6, 8, split (8,8)
constexpr uint32_t kMaskRefine = 0x38000;  // fp64 distance re-evaluation: split classes only (latency matters)

// resident CTAs per SM the pair kernels are compiled for (register budget via __launch_bounds__)
QP_HD2 int ctas_per_sm(int C, int W, bool fp64) {
    if (W > 1) return fp64 ? 1 : (C <= 8 ? 3 : 2);
    return fp64 ? (C <= 4 ? 3 : 2) : (C <= 6 ? 4 : (C <= 12 ? 3 : 2));
}
// pairs in flight per CTA
QP_HD2 int units_per_cta(int W) { return W == 1 ? kWarpsPerCta : 1; }

struct alignas(16) PairInfo {
    int64_t xoff, yoff;   // start of the row / column sequence in d_seqs
    int32_t n, m;         // rows (first sequence), columns (second sequence)
    int16_t cls;          // class index, -1 = skipped (invalid pair)
    int16_t nb;           // column blocks of 32*C columns
    int32_t bin;          // size bin of its scratch slot
};

// ---- per-pair scratch slot ---------------------------------------------------------------------------------
// block b, step t:  F planes | [32] int2 exponents (e_hmm, e_pf), one per lane
//   fp32: [ceil(C/2)][32] float4 = (F_hmm, F_pf) of the lane's columns 2u and 2u+1  (every warp access is 512 B contiguous)
//   fp64: [C][32] double2  = (F_hmm, F_pf) of the lane's column k
// The exponent record of a step is written (and read back) only on the last step of every renormalisation period
// and on the last step of the block: a lane's exponents cannot change in between.
// The backward pass reuses consumed step records as per-row entry buffers: the kept (value, column) entries of
// row i (found by lane l at step i+l, highest columns first) go to the F area of step record i+32, which every
// lane has consumed before the first of them is written; row i's entry count goes to rowcnt[b][i]. Sparsification
// therefore adds one step record and 4 bytes per row of scratch.
QP_HD2 int f_units(int C, int real_bytes) { return real_bytes == 4 ? (C + 1) / 2 : C; }   // 16-byte words per lane and step
QP_HD2 int64_t exps_offset(int C, int real_bytes) { return (int64_t)f_units(C, real_bytes) * 512; }
QP_HD2 int64_t step_stride(int C, int real_bytes) { return exps_offset(C, real_bytes) + 256; }
QP_HD2 int num_steps(int n) { return n + 33; }
QP_HD2 int64_t bnd_rec_bytes(int real_bytes) { return 12 * (int64_t)real_bytes + 16; }   // see BndRec in qp_pair.cuh
// byte offset of rowcnt[nb][n+1] (int32) inside the slot
QP_HD2 int64_t rowcnt_offset(int n, int C, int nb, int real_bytes) {
    int64_t b = (int64_t)nb * num_steps(n) * step_stride(C, real_bytes);
    if (nb > 1) b += 2 * (int64_t)(n + 1) * bnd_rec_bytes(real_bytes);
    return (b + 15) & ~(int64_t)15;
}
QP_HD2 int64_t slot_bytes(int n, int C, int nb, int real_bytes) {
    int64_t b = rowcnt_offset(n, C, nb, real_bytes) + (int64_t)nb * (n + 1) * 4;
    return (b + 255) & ~(int64_t)255;
}

// choose the class of a pair with n rows and `cols` = m+1 columns among the classes of `mask`:
//   1. the narrowest packed class whose single block holds all columns (least padding, one warp per pair);
//   2. else, for pairs of moderate size, the narrowest two-block class that holds the columns: one warp per pair keeps
//      the efficiency of the packed classes (no idle warp, no ring hand-off: a packed class alone moves 4.8 TB/s of
//      DRAM traffic, the 4-warp split class for 513..768 columns 2.0); the size limit keeps the time a single warp
//      spends on one pair (~8 ns per cell) well below the time of a call that contains such pairs;
//   3. else the split class with the shortest pipeline: passes * (rows + 32 * active warps) * (C + per-step overhead
//      expressed in cells), a pass = W neighbouring blocks;
// Returns the class index (-1 if the mask holds no class that can take the pair) and the number of 32*C-column blocks.
constexpr int64_t kTwoBlockMaxCells = 400000;
constexpr int kMultiBlockMaxRows = 256;
QP_HD2 int choose_class(int n, int cols, uint32_t mask, bool fp64, int* nb_out) {
    constexpr int kStepOverhead = 6;
    int best = -1, best_nb = 0;
    int64_t best_cost = 0;
    for (int c = 0; c < kNumPacked; ++c) {
        const int C = class_C(c, fp64);
        if (!((mask >> c) & 1) || C == 0) continue;
        if (cols <= 32 * C) {
            *nb_out = 1;
            return c;
        }
    }
    if ((int64_t)n * cols <= kTwoBlockMaxCells)
        for (int c = kSplitEnd; c < kNumClasses; ++c) {
            const int C = class_C(c, fp64);
            if (!((mask >> c) & 1) || C == 0) continue;
            if (cols <= 64 * C) {
                *nb_out = 2;
                return c;
            }
        }
    // 2b. short rows against many columns (at most kMultiBlockMaxRows rows): the ramp of a split pass (32 steps per
    //     active warp) would outweigh the rows; one warp runs the column blocks of the widest multi-block class one
    //     after the other instead (n + 32 steps per block)
    if (n <= kMultiBlockMaxRows && (int64_t)n * cols <= kTwoBlockMaxCells && ((mask >> (kNumClasses - 1)) & 1)) {
        const int C = class_C(kNumClasses - 1, fp64);
        if (C > 0) {
            *nb_out = (cols + 32 * C - 1) / (32 * C);
            return kNumClasses - 1;
        }
    }
    for (int c = kNumPacked; c < kSplitEnd; ++c) {
        if (!((mask >> c) & 1)) continue;
        const int C = class_C(c, fp64), W = class_W(c, fp64);
        const int nb = (cols + 32 * C - 1) / (32 * C);
        const int act = nb < W ? nb : W;
        const int64_t cost = (int64_t)((nb + W - 1) / W) * (n + 1 + 32 * act) * (C + kStepOverhead);
        if (best < 0 || cost < best_cost) {
            best = c;
            best_nb = nb;
            best_cost = cost;
        }
    }
    *nb_out = best_nb;
    return best;
}

// size bins: 8 per octave. bin_of(v) for v >= 16; bin_ub = exclusive upper bound of the bin's range.
QP_HD2 int bin_of(uint64_t v) {
    int e = 63;
    while (e > 3 && !((v >> e) & 1)) --e;
    int mant = (int)((v >> (e - 3)) & 7);
    int b = (e - 3) * 8 + mant;
    return b < kNumBins ? b : kNumBins - 1;
}
QP_HD2 uint64_t bin_ub(int b) {
    int e = b / 8 + 3, mant = b % 8;
    return (uint64_t)(8 + mant + 1) << (e - 3);
}

// fp64 distance re-evaluation queue, one list per split fp64 class (kMaskRefine). The fp32
// pair kernels append the pairs whose fp32 distance is below the limit; two sets of fp64 kernels consume the lists
// through one cursor per class:
//   pollers  a few CTAs per class, launched with the fp32 classes (after them, so they take SM room only when the fp32
//            kernels leave some): they wait for entries to appear, claim a position only when its entry is visible,
//            and leave when every fp32 CTA has finished and the list is drained -- or after kPollIdleMax empty polls in
//            a row, so that no number of calls in flight can keep every SM busy with waiting CTAs (qp_kernel.cuh).
//            Their scratch slots are reserved at schedule time, sized for the largest pair the class could receive.
//   drainers full-width kernels launched after the fp32 classes have joined, for what is left; slots from the fp32
//            slot region, sized for the largest pair actually queued.
constexpr int kPollCtas = 32;         // most pollers per class; poll_ctas() scales it to the device
constexpr int kPollIdleMax = 8192;    // empty polls in a row (2 us apart, ~20 ms) after which a poller leaves
// pollers per class on a device of `sms` SMs: the three fp64 classes together never ask for more than 2/3 of them
__host__ __device__ constexpr int poll_ctas(int sms) { return sms * 2 / 9 < 1 ? 1 : (sms * 2 / 9 < kPollCtas ? sms * 2 / 9 : kPollCtas); }
constexpr int kListPad = 1024;        // every DRAINER CTA pulls one index past the end of its list: the drainer grid is
                                      // clamped to this (qp_api.cu); pollers claim only filled positions
struct RefineQ {
    int32_t count[kNumClasses];                   // pairs queued, per fp64 class
    int32_t cursor[kNumClasses];                  // next list position to consume
    int32_t possible[kNumClasses];                // pairs of the call that WOULD go to the class (schedule time)
    int32_t Wpoll[kNumClasses];                   // pollers granted
    unsigned long long poll_slot_bytes[kNumClasses];   // largest fp64 scratch slot among all pairs of the class
    unsigned long long poll_slot0[kNumClasses];
    int32_t W[kNumClasses];                       // drainers granted
    unsigned long long slot_bytes[kNumClasses];   // largest fp64 scratch slot among the queued pairs
    unsigned long long slot0[kNumClasses];        // byte offset of the class's first slot inside the slot region
};

struct SchedHeader {
    int32_t status[4];                       // mirrors qp_output.status
    unsigned long long pool_cursor;          // CSR staging pool bump pointer (entries)
    int32_t cls_count[kNumClasses];          // pairs per class
    int32_t cls_start[kNumClasses];          // start of the class in order[]
    int32_t cls_W[kNumClasses];              // resident warps (= scratch slots) granted to the class
    int32_t cls_slot0[kNumClasses];          // first entry of the class in slot_off[]
    int32_t cls_cursor[kNumClasses];         // next position in the class's order list
    RefineQ rq;
    unsigned long long poll_bytes;           // head of the slot region, reserved for the pollers' slots
    int32_t producers_done;                  // fp32 class CTAs that have exited
    int32_t pad_;
    uint32_t hist[kNumClasses][kNumBins];    // pairs per (class, size bin)
    uint32_t bin_start[kNumClasses][kNumBins];   // position of the bin inside the class, largest bins first
    uint32_t bin_fill[kNumClasses][kNumBins];
};

// kernel argument block (passed by value, __grid_constant__)
template <typename R> struct KArgs {
    typename Traits<R>::vec2 tab[kTabDim * kTabDim];   // (em_hmm, em_pf)[x*32+y], sentinel row/col zero
    Weights<R> wh, wp;
    W2 w2;                       // fp32: (hmm, pf) weight pairs for the packed recurrences (qp_both.cuh)
    R tau;
    int rescale_mask;            // renormalise every (mask+1) steps
    int32_t k;                   // number of sequences (dist is k x k)
    int32_t refine_pass;         // 0: class lists; 1 / 2: poller / drainer of the fp64 re-evaluation queue, distances only
    int32_t producers_total;     // fp32 class CTAs of the call (pollers leave when all of them have exited); 0: not counted
    float refine_below;          // fp32 pass: queue pairs whose distance is below this (<=0: never)
    double lx_h[kTabDim], lx_p[kTabDim];   // insert log-weights (for the logZ constant)
    const uint8_t* seqs;
    const int32_t* pairs;        // [P][2]
    const PairInfo* info;
    const int32_t* order;
    SchedHeader* hdr;
    const int64_t* slot_off;     // byte offset of each slot inside slots
    char* slots;
    int32_t* refine_list;        // [3 split classes][refine_stride] pair indices queued for fp64 re-evaluation, -1 = empty
    int64_t refine_stride;
    uint32_t refine_cmask;       // classes of the fp64 distance re-evaluation
    // outputs
    const int64_t* pair_row_base;
    int32_t* row_ptr;
    float2* pool;                // CSR staging pool: (value, column bits) per entry, completion order
    int64_t pool_cap;
    int32_t* nnz;                // per pair
    int64_t* pool_off;           // per pair
    float* dist;
    float* dense_P;
    const int64_t* dense_off;
    double* logZ;
    // memory-limited mode (qp_posteriors_budgeted): histogram of the kept posterior values over threshold bins
    unsigned long long* tau_hist;   // [kTauBins] or nullptr
    int32_t tau_bits0;              // bit pattern of the threshold as a float: bin = (bits(P) - tau_bits0) >> kTauShift
};

// threshold bins of the memory-limited mode: 16 per octave above the requested threshold (positive floats order like
// their bit patterns, so a bin is a range of bit patterns); the last bin is open-ended
constexpr int kTauBins = 128;
constexpr int kTauShift = 19;

}  // namespace qp
