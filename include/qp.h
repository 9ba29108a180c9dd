/*
 * qp.h -- C ABI of libqp.so: B200-native (sm_100a) all-pairs posterior stage of QuickProbs 2.
 *
 * What it computes (Methods, stage I): "Posterior probability matrices are calculated for all
 * sequence pairs on the basis of hidden Markov model and partition function. The matrices are further employed
 * to establish maximum expected accuracy alignments. Alignment scores are used to estimate pairwise distances".
 * The matrices are kept "in a sparse form" (footnote). The paper prints no recurrence or constant;
 * the exact definitions are the readings of SURVEY.md section 8(c) (c-1 model, c-2 combine/threshold/MEA/distance),
 * restated in DESIGN.md. Every step (schedule, forward, backward, combine, sparsify, expected accuracy) runs in
 * CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *  - "d_" pointers are DEVICE pointers owned by the caller (e.g. torch tensors); "h_"/struct pointers are HOST.
 *  - The library allocates no device memory: scratch comes from the caller's workspace.
 *  - Work is enqueued on `cuda_stream` (a cudaStream_t passed as void*). With QP_FLAG_SYNC_STATUS the call
 *    synchronises the stream once at the end, reads the device status word and returns it; without it the call
 *    returns after enqueueing and device-detected errors are only visible in qp_output.status.
 *  - Return value: 0 (QP_OK) or a negative QP_ERR_* code. No exception or abort crosses the ABI.
 *  - Rows of pair p's matrix = residues of the FIRST index of d_pairs[p]; columns = residues of the second.
 */
#ifndef QP_H_
#define QP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QP_MAX_INS 2
#define QP_MAX_ALPHABET 31 /* residue codes 0..alphabet-1; code 31 is reserved internally */
#define QP_MAX_LEN 65535   /* longest supported sequence (CSR scratch packs a column offset in 16 bits) */

enum {
    QP_OK = 0,
    QP_ERR_INVALID_ARG = -1,        /* NULL pointer, bad alphabet / n_ins / threshold / precision, P or k < 0  */
    QP_ERR_BAD_RESIDUE = -2,        /* a residue code >= alphabet                (device-detected)              */
    QP_ERR_EMPTY_SEQUENCE = -3,     /* a listed sequence has length 0 or > QP_MAX_LEN (device-detected)         */
    QP_ERR_BAD_PAIR = -4,           /* pair index out of [0,k) or x == y          (device-detected)              */
    QP_ERR_WORKSPACE_TOO_SMALL = -5,/* workspace cannot hold the fixed arrays + one scratch slot per class     */
    QP_ERR_NNZ_CAPACITY = -6,       /* CSR needs more than nnz_capacity entries; pair_nnz_base[P] = required   */
    QP_ERR_CUDA = -7,               /* a CUDA runtime call failed                                              */
    QP_ERR_RANGE = -8,              /* model weights outside the dynamic range the kernels renormalise for     */
    QP_ERR_STATIC_LIMIT = -9        /* qp_guide_tree_static: k > QP_GUIDE_TREE_STATIC_MAX_K (built-in scratch)   */
};

enum { QP_FP32 = 0, QP_FP64 = 1 };

enum {
    QP_FLAG_SYNC_STATUS = 1,        /* synchronise the stream at the end and return the device status          */
    QP_FLAG_NO_REFINE = 2,          /* QP_FP32 only: skip the fp64 re-evaluation of near-identical pairs        */
    QP_FLAG_NO_POLLERS = 4          /* QP_FP32 only: run the fp64 re-evaluation only AFTER the fp32 kernels (drainers), not
                                       also beside them (pollers). Pollers are kernels that wait, on the device, for the
                                       fp32 kernels of the same call to queue pairs. They never block progress: a poller
                                       claims only entries that are already visible and leaves after ~20 ms without
                                       work, whatever else shares the device. But with several calls in flight on
                                       different streams the waiting kernels of one call sit in front of the next call's
                                       kernels in the hardware queues they share and cost throughput: such callers
                                       (qp_posteriors_host does) should set this flag                               */
};

/*
 * One weighted pair automaton, natural-log weights. States M, X_1..X_G, Y_1..Y_G;
 * X/Y symmetric by construction; no X<->Y transition. -INFINITY is a legal weight (probability 0).
 *   HMM instance: log_match = ln e(a,b), log_ins = ln q(a), t_MI = ln delta_g, t_II = ln eps_g,
 *                 t_IM = ln(1-eps_g), t_MM = ln(1-2 sum delta), init/end = ln pi.
 *   PF instance (substitution matrix, gap penalties, temperature), passed already divided by T:
 *                 log_match = s(a,b)/T, log_ins = 0, t_MM = t_IM = 0, t_MI = init_I = -g_open/T, t_II = -g_ext/T,
 *                 init_M = end = 0.
 */
typedef struct {
    int32_t n_ins;           /* G: 1 or 2                                                   */
    int32_t alphabet;        /* A: 2..QP_MAX_ALPHABET, the same for both models             */
    const double* log_match; /* host, A*A row-major, must be symmetric                      */
    const double* log_ins;   /* host, A                                                     */
    double t_MM, t_MI[QP_MAX_INS], t_II[QP_MAX_INS], t_IM[QP_MAX_INS];
    double init_M, init_I[QP_MAX_INS], end_M, end_I[QP_MAX_INS];
} qp_model;

typedef struct {
    qp_model hmm, pf;
    double threshold;        /* tau > 0: CSR keeps P(i,j) >= tau (value from BASELINE.json)        */
    int32_t precision;       /* QP_FP32 | QP_FP64: arithmetic of the DP kernels                                */
    int32_t flags;           /* QP_FLAG_*                                                                      */
    double refine_below;     /* QP_FP32: pairs whose fp32 distance is below this are re-evaluated in fp64
                                (distance only). <= 0 selects the default 0.25; for pairs with n + m > 4000 the
                                limit is scaled by sqrt((n + m) / 4000). See DESIGN.md "Distances".             */
} qp_params;

/* Outputs. All device memory, caller-allocated. Optional members may be NULL. */
typedef struct {
    int64_t* pair_row_base;  /* [P+1] exclusive prefix of (n_p+1): pair p's row_ptr starts here                 */
    int64_t* pair_nnz_base;  /* [P+1] exclusive prefix of nnz_p:   pair p's col_idx/val start here              */
    int32_t* row_ptr;        /* [sum(n_p+1)] offsets local to the pair (0..nnz_p)                               */
    int32_t* col_idx;        /* [nnz_capacity] 0-based column (residue of the second sequence), ascending/row  */
    float* val;              /* [nnz_capacity] combined posterior P(i,j) >= tau                                 */
    int64_t nnz_capacity;
    float* dist;             /* [k*k] row-major; (x,y) and (y,x) are written for listed pairs only              */
    float* dense_P;          /* optional: concatenated dense n_p*m_p row-major matrices, pair order (tests)    */
    double* logZ;            /* optional [P][4]: ln Z of hmm fwd, hmm bwd, pf fwd, pf bwd                        */
    int32_t* status;         /* [4] device status word: {code, pair index or -1, detail, pairs whose distance was
                                re-evaluated in fp64 (those whose fp32 distance came out below refine_below)}       */
} qp_output;

/*
 * Host-only query (no device access): bytes of workspace that let every scheduling class run with its full
 * complement of resident warps, capped at budget_bytes (0 = no cap). Never less than the minimum that
 * qp_posteriors accepts for this input. h_offsets [k+1], h_pairs [P][2] are host copies of the device inputs.
 * Errors: QP_ERR_INVALID_ARG, QP_ERR_BAD_PAIR, QP_ERR_EMPTY_SEQUENCE, QP_ERR_WORKSPACE_TOO_SMALL (budget below
 * the minimum; *out_bytes then holds the minimum).
 */
int qp_workspace_bytes(const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P,
                       const qp_params* params, int64_t nnz_capacity, int want_dense, size_t budget_bytes,
                       size_t* out_bytes);

/*
 * The hot path. d_seqs: packed residue codes (uint8); d_offsets [k+1]: sequence s is
 * d_seqs[d_offsets[s] .. d_offsets[s+1]); d_pairs [P][2] int32. Steps, all on the device:
 *   a0 schedule (length classes: short pairs packed one per warp, long pairs split over the warps of a CTA;
 *      largest-first order, scratch slots)
 *   a1-a4 pair-HMM and partition-function forward and backward
 *   a5 combine P = sqrt((P_hmm^2+P_pf^2)/2), a6 threshold + CSR compaction
 *   a7 expected-accuracy (MEA) max-plus DP and d = 1 - A(n,m)/min(n,m)
 * d_workspace must be 256-byte aligned. Outputs for pairs after an error are unspecified.
 */
int qp_posteriors(const uint8_t* d_seqs, const int64_t* d_offsets, int32_t k, const int32_t* d_pairs, int64_t P,
                  const qp_params* params, void* d_workspace, size_t workspace_bytes, const qp_output* out,
                  void* cuda_stream);

/*
 * The posterior stage on HOST buffers (BASELINE.json configs[3]: "memory-budgeted by streaming pair batches"): inputs
 * and outputs live in host memory (pin them -- cudaHostAlloc / cudaHostRegister -- or the copies will not overlap
 * anything). The pair list is cut into batches of about a quarter of the family (4e8 .. 6e9 cells), shrunk until two
 * batches fit d_workspace; every batch goes through qp_posteriors; two batches are in flight, so that the CSR of one
 * travels back over PCIe while the kernels of the next run. A batch that turns out denser than beta_guess is split in
 * two and run again. The call returns when every output is in host memory (it synchronises).
 *   h_seqs / h_offsets / h_pairs   as d_seqs / d_offsets / d_pairs of qp_posteriors, in host memory
 *   d_workspace                    DEVICE memory, 256-byte aligned, caller-owned; holds the device copies of the inputs,
 *                                  the k x k distance matrix, and per batch in flight the outputs and the workspace of
 *                                  qp_posteriors. qp_posteriors_host_workspace_bytes gives the size at which no batch has
 *                                  to be shrunk; less works down to one pair per batch
 *   out                            host arrays laid out like qp_output -- pair order, global prefixes; beta_guess: expected
 *                                  nnz / cells (<= 0: 0.05) sizes the per-batch device CSR; the call fills status,
 *                                  h2d_bytes / d2h_bytes (bytes it copied) and batches
 * Returns QP_OK or an error of qp_posteriors; QP_ERR_NNZ_CAPACITY if out->nnz_capacity is too small (pair_nnz_base[P] =
 * entries required). A batch denser than beta_guess is split in two and taken again; a SINGLE pair whose entries do not
 * fit the per-batch device CSR ends the call with QP_ERR_NNZ_CAPACITY and status[1] = that pair (raise beta_guess).
 * params->flags: QP_FLAG_NO_REFINE is honoured, the others are set by the call (it runs its batches with
 * QP_FLAG_NO_POLLERS).
 */
typedef struct {
    int64_t* pair_row_base;  /* [P+1] */
    int64_t* pair_nnz_base;  /* [P+1] */
    int32_t* row_ptr;        /* [sum(n_p+1)] */
    int32_t* col_idx;        /* [nnz_capacity]; not written (may be NULL) when col_idx16 is given */
    float* val;              /* [nnz_capacity] */
    int64_t nnz_capacity;
    float* dist;             /* [k*k] */
    uint16_t* col_idx16;     /* optional [nnz_capacity]: the columns as 16-bit values instead (lossless, QP_MAX_LEN is
                                65535): 6 instead of 8 bytes per entry cross PCIe, which is what bounds this call */
    double beta_guess;       /* in */
    int32_t status[4];       /* out: {code, pair index or -1, detail, pairs re-evaluated in fp64} */
    int32_t batches;         /* out */
    int32_t reserved;
    int64_t h2d_bytes, d2h_bytes;   /* out */
} qp_host_output;
int qp_posteriors_host_workspace_bytes(const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P,
                                       const qp_params* params, double beta_guess, size_t* out_bytes);
int qp_posteriors_host(const uint8_t* h_seqs, const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P,
                       const qp_params* params, void* d_workspace, size_t workspace_bytes, qp_host_output* out,
                       void* cuda_stream);

/*
 * Memory-limited mode ("fit analysis in user-specified amount of RAM by decreasing sparsity coefficient in
 * posterior matrices"; memory for the posterior matrices limits the set size). The caller's CSR capacity
 * out->nnz_capacity is the budget (8 bytes per entry). At most TWO passes of the stage:
 *   pass 1  qp_posteriors at params->threshold; on the way every kept value is counted into threshold bins (16 per
 *           octave above the threshold). If the CSR fits, that is the result (*passes = 1).
 *   pass 2  otherwise the smallest bin edge tau' whose count of values >= tau' fits the capacity is taken from the
 *           histogram -- exactly, since the second pass recomputes the very same values -- and the stage is run again
 *           at tau' (*passes = 2).
 * On success *tau_used is the threshold the returned CSR was cut at; every output is exactly what qp_posteriors
 * returns for that threshold. Synchronises the stream after every pass. Returns QP_ERR_NNZ_CAPACITY if max_passes is 1
 * and the CSR does not fit, or if not even the top bin fits (pair_nnz_base[P] = entries required at the last threshold
 * tried, *tau_used = that threshold); any other error of qp_posteriors unchanged. tau_used and passes are HOST
 * pointers (may be NULL).
 * qp_last_tau_curve: the histogram of the last qp_posteriors_budgeted call of this thread as a curve: tau[b] = lower
 * edge of bin b (tau[0] = the requested threshold), count[b] = kept values >= tau[b] (so count[b] / cells is the
 * sparsity coefficient beta at threshold tau[b]). Returns the number of bins written (<= max_bins, 128
 * in all) or QP_ERR_INVALID_ARG if there is no histogram. HOST pointers.
 */
int qp_posteriors_budgeted(const uint8_t* d_seqs, const int64_t* d_offsets, int32_t k, const int32_t* d_pairs, int64_t P,
                           const qp_params* params, void* d_workspace, size_t workspace_bytes, const qp_output* out,
                           void* cuda_stream, int max_passes, double* tau_used, int* passes);
int qp_last_tau_curve(double* tau, int64_t* count, int max_bins);

/*
 * Stage II ("pairwise distances ... are given as an input for weighted UPGMA
 * algorithm for guide tree construction"; tree-guided distance = "a number of nodes in a minimal
 * subtree containing both x and y", Figure 2).
 *   d_dist     [k*k] fp32, symmetric, entries >= 0 (the matrix qp_posteriors wrote); only i != j is read
 *   d_merge    [k-1][2] node ids of the two children of merge t (leaves 0..k-1, the node made by merge t is k+t);
 *              the child that lived in the smaller slot first
 *   d_height   [k-1] distance at which merge t happened (non-decreasing)
 *   d_leaves   [2k-1] leaf count of every node;  d_parent [2k-1] parent node id, -1 for the root
 *   d_treedist optional [k*k] int32: 2*leaves(lca(x,y)) - 1, diagonal 1 (NULL: not computed)
 * Weighted UPGMA: merge the closest pair of clusters (ties: the lexicographically smallest slot pair i < j, a cluster
 * keeps the slot of its smaller-slot child), d(u,m) = (d(i,m) + d(j,m)) / 2 evaluated in fp32. All device pointers
 * are caller-owned; the workspace holds a working copy of the matrix and the per-row nearest neighbours
 * (qp_guide_tree_workspace_bytes). Work is enqueued on the stream, nothing is synchronised.
 * Errors: QP_ERR_INVALID_ARG (NULL pointer, k < 1, workspace too small or misaligned), QP_ERR_CUDA.
 */
size_t qp_guide_tree_workspace_bytes(int32_t k);
int qp_guide_tree(const float* d_dist, int32_t k, int32_t* d_merge, float* d_height, int32_t* d_leaves,
                  int32_t* d_parent, int32_t* d_treedist, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * qp_guide_tree without a workspace argument and without any allocation, for callers that cannot allocate device
 * memory: a plug-in inside a host application that owns the whole device heap and hands out only input and output
 * buffers; a step inside a latency-critical loop, where cudaMalloc / cudaFree may block on the driver and synchronise
 * the device; a process held to a fixed memory reservation on a shared GPU, where a late allocation can fail even
 * though the inputs fit. Same arguments, same kernels and bit-identical outputs as qp_guide_tree, minus d_workspace:
 * the scratch of the merge loop is an array built into libqp.so.
 *   limit      k <= QP_GUIDE_TREE_STATIC_MAX_K (1024: BASELINE.json's largest family has 1000 sequences). Larger k
 *              returns QP_ERR_STATIC_LIMIT and launches nothing; use qp_guide_tree with your own workspace.
 *   cost       the array (QP_GUIDE_TREE_STATIC_BYTES, about 4 MiB) is part of the library image: every GPU on which
 *              libqp.so's kernels are loaded holds it until the process exits, whether or not this call is used.
 *   first call the first call on each device looks up the array's device address (one cudaGetSymbolAddress with that
 *              device current; result kept for the life of the process). Make that first call outside any stream
 *              capture, with the device you mean to use current.
 *   sharing    every call on a device uses the SAME array. Calls on one stream run in order and are fine. Two calls
 *              that can overlap on the GPU (different streams, different host threads without ordering) race on it
 *              and give wrong trees: order them yourself (one stream, or events). Nothing has to be cleared between
 *              calls -- the merge kernel rewrites every scratch word it later reads -- so a call never sees what the
 *              previous one left, whatever its k was.
 * The call runs no cudaMalloc, cudaFree or allocating library routine; it enqueues two kernels on the stream and
 * returns without synchronising. Other errors: QP_ERR_INVALID_ARG (NULL pointer, k < 1), QP_ERR_CUDA (no current
 * device, address lookup or launch failed).
 */
#define QP_GUIDE_TREE_STATIC_MAX_K 1024
#define QP_GUIDE_TREE_STATIC_BYTES (QP_GUIDE_TREE_STATIC_MAX_K * (QP_GUIDE_TREE_STATIC_MAX_K * 4 + 8 + 4 + 1))
int qp_guide_tree_static(const float* d_dist, int32_t k, int32_t* d_merge, float* d_height, int32_t* d_leaves,
                         int32_t* d_parent, int32_t* d_treedist, void* cuda_stream);

/*
 * Stage III: selective consistency transformation of the sparse posterior matrices.
 * "consistency relies on the relaxation of posterior probability matrices by other sequences";
 * PAPER.md:55, :63 (Figure 2): "posterior matrix S_xy is relaxed over sequence z if assumed function f(d_xz, d_yz)
 * fulfills given condition", d = the tree-guided distance, thresholded deterministically: f(d_xz, d_yz) <= T
 * (best setting: maximum, T ~ 200); S_xy is amplified by h_xy, which "varies from 1
 * when no relaxations of S_xy are performed, to h when maximum number of relaxations ... is done (200 in our case)",
 * best h = 3; PAPER.md:59 footnote: the matrices are sparse. The paper prints no formula; the reading
 * (the oracle oracle/qp_consistency.py follows the same):
 *     sel(x,y) = { z != x, y : both pairs {x,z}, {z,y} are in the input and f(treedist[x][z], treedist[y][z]) <= T }
 *     h_xy     = 1 + (h - 1) * min(|sel|, max_relax) / max_relax
 *     S'_xy    = ( 2 h_xy S_xy + sum_{z in sel(x,y)} S_xz S_zy ) / ( 2 h_xy + |sel(x,y)| ),  S_zx = S_xz^T,
 *                evaluated on the cells stored in S_xy only; values below `threshold` are dropped.
 * Every relaxed matrix is computed from the INPUT matrices (one transformation = one call; 2 calls for
 * k < 50, 1 otherwise -- qp_consistency_passes). Arithmetic: fp32, fixed summation order (reproducible).
 *   in       the per-pair CSR that qp_posteriors wrote (same d_offsets / d_pairs); an unordered pair should be
 *            listed once
 *   nnz      HOST value: entries of the input, in->pair_nnz_base[P]
 *   out      pair_nnz_base [P+1], row_ptr [sum(n_p+1)] (same row layout as the input: in->pair_row_base serves both),
 *            col_idx / val [nnz_capacity]; nnz_capacity >= nnz always suffices (the pattern only shrinks);
 *            relaxations: optional [P], |sel| of every pair; status [4] device status word {code, pair or -1, 0, 0}
 * Errors: QP_ERR_INVALID_ARG; device-detected in out->status: QP_ERR_BAD_PAIR, QP_ERR_EMPTY_SEQUENCE,
 * QP_ERR_WORKSPACE_TOO_SMALL, QP_ERR_NNZ_CAPACITY. Work is enqueued on the stream, nothing is synchronised. All
 * device buffers are caller-owned; the workspace (qp_consistency_workspace_bytes, a host-only query on host copies
 * of the offsets and pairs) holds the pair lookup table, interleaved copies of every matrix and of its transpose,
 * and the staging area of the relaxed entries.
 */
enum { QP_SEL_MAX = 0, QP_SEL_MIN = 1, QP_SEL_SUM = 2 };
typedef struct {
    int32_t T;               /* selection threshold on f(treedist[x][z], treedist[y][z])                        */
    int32_t f;               /* QP_SEL_MAX (the paper's best), QP_SEL_MIN or QP_SEL_SUM                          */
    double h;                /* amplification of the original signal at max_relax relaxations, >= 1 (paper: 3)   */
    int32_t max_relax;       /* relaxations at which h_xy reaches h (paper: 200)                                 */
    int32_t reserved;
    double threshold;        /* relaxed values below it are dropped (stage I's tau)                              */
} qp_consistency_params;
typedef struct {             /* per-pair CSR matrices, device, layout of qp_output                               */
    const int64_t* pair_row_base;
    const int64_t* pair_nnz_base;
    const int32_t* row_ptr;
    const int32_t* col_idx;
    const float* val;
} qp_csr;
typedef struct {
    int64_t* pair_nnz_base;
    int32_t* row_ptr;
    int32_t* col_idx;
    float* val;
    int64_t nnz_capacity;
    int32_t* relaxations;    /* optional */
    int32_t* status;
} qp_csr_out;
int qp_consistency_workspace_bytes(const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P, int64_t nnz,
                                   size_t* out_bytes);
int qp_consistency(const int64_t* d_offsets, int32_t k, const int32_t* d_pairs, int64_t P, const qp_csr* in, int64_t nnz,
                   const int32_t* d_treedist, const qp_consistency_params* params, void* d_workspace,
                   size_t workspace_bytes, const qp_csr_out* out, void* cuda_stream);
/* "the number of transformations is adjusted to the number of sequences (2 for k < 50, 1 otherwise)". */
int qp_consistency_passes(int32_t k);

/* Number of kernels the last qp_posteriors call on this thread launched (bench.py's gpu_launches). */
int qp_last_launch_count(void);

/*
 * Phase timing for bench.py's roofline line. qp_set_profile(1) makes later qp_posteriors calls on this thread
 * record CUDA events on the caller's stream at the phase boundaries (no synchronisation is added). After the
 * caller has synchronised the stream, qp_get_profile fills ms[0..3] with the device time of the last call:
 *   ms[0] schedule (a0), ms[1] pair kernels (a1-a7, all classes, fork to join; the pollers of the fp64 distance queue
 *   run beside them), ms[2] what is left after their join: the drainers of the fp64 distance queue (pairs the pollers
 *   had not taken) and the CSR placement (scan + copy) beside them, the pollers' tail if any, ms[3] status word.
 * Returns QP_OK, or QP_ERR_INVALID_ARG if no profiled call has completed.
 */
void qp_set_profile(int on);
int qp_get_profile(float ms[4]);
/* Per scheduling class c: start and stop of its pair kernel in ms after the end of the schedule phase, -1 for classes
 * that did not run. Same preconditions as qp_get_profile.
 *   0..14   packed: one warp per pair, stripe width C = c + 2, at most 32 C columns (one column block)
 *   15..17  split: the 4 warps of a CTA share one long pair (C = 8, 12, 16)
 *   18..21  packed multi-block: one warp per pair, C = c - 18 + 9, the column blocks of 32 C columns one after the other.
 *           Takes pairs of 513..768 columns (two or three blocks) and, in class 21, every pair of at most 256 rows and
 *           4e5 cells whatever its width (up to ~170 blocks): a split pass would spend more on its ramp than on the rows */
#define QP_NUM_CLASSES 22
int qp_get_profile_classes(float start_ms[QP_NUM_CLASSES], float stop_ms[QP_NUM_CLASSES]);

/*
 * Releases what the library keeps per host thread and device between calls: the side streams and events that fork
 * and join the per-class kernels (created lazily by the first qp_posteriors call of a thread on a device). Call it
 * from the thread that made the calls, after its streams have been synchronised. Later calls re-create them. A thread
 * that exits without calling it releases them on its way out (the work it enqueued should have been synchronised).
 */
void qp_shutdown(void);

/*
 * Measured arithmetic peaks of the current device, for the roofline lines of bench.py ("measure it
 * with a ... micro-benchmark at the sustained clock"; "report the FP32-pipe bound beside it"). Three micro-kernels of
 * independent dependency chains, 32 warps per SM, a few ms each, best of two timed repetitions:
 *   ffma_per_s        scalar fp32 FMA lane-operations per second (FFMA);  / 32 = warp instructions per second when
 *                     nothing but the issue slots limits a kernel (warp_instr_per_s)
 *   ffma2_fma_per_s   scalar-equivalent FMAs per second through the packed instruction (fma.rn.f32x2 -> FFMA2), the
 *                     one the pair kernels use for the two automata side by side
 *   mufu_per_s        sqrt.approx per second (MUFU pipe; the pair kernels issue one per cell)
 * d_scratch: at least sms * 4096 bytes of device memory (caller-owned). Synchronises the stream. Errors:
 * QP_ERR_INVALID_ARG, QP_ERR_WORKSPACE_TOO_SMALL, QP_ERR_CUDA.
 */
typedef struct {
    int32_t sms;
    int32_t reserved;
    double ffma_per_s, ffma2_fma_per_s, mufu_per_s, warp_instr_per_s;
} qp_peaks;
int qp_measure_peaks(qp_peaks* out, void* d_scratch, size_t scratch_bytes, void* cuda_stream);

const char* qp_status_string(int status);
const char* qp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QP_H_ */
