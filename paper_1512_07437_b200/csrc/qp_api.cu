// qp_api.cu -- host side of the C ABI (include/qp.h) plus the small device-side scheduling kernels.
//
// Schedule ("redesigning graphics processor calculations to handle sequences of
// any length ... more efficient memory allocation model"): everything below runs on the device, the host never
// sees a sequence length.
//   classify : per pair -> (rows n, cols m, class: packed stripe width or split (C, W), scratch bytes -> size bin);
//              histogram per class/bin
//   bins     : per class, bins ordered largest first -> start position of every bin
//   scatter  : counting sort of the pair indices into order[] (class-major, largest scratch first)
//   slots    : grant W_c resident warps per class under the workspace budget; warp w's scratch slot is sized for
//              the w-th largest pair of its class, which bounds every pair that warp will pull later
//   scans    : pair_row_base (CSR row_ptr placement), dense offsets, and after the pair kernels pair_nnz_base
//   copy     : staging pool (completion order) -> caller's col_idx/val in pair order
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>
#include <algorithm>

#include "qp.h"
#include "qp_internal.h"
#include "qp_scan.cuh"

namespace qp {

enum : int { kModeCsr = 0, kModeFull = 1, kModeDist = 2 };   // see qp_pair.cuh
template <typename R, int GP, int C, int MODE, int W> cudaError_t launch_pair(const KArgs<R>& ka, int grid, cudaStream_t st);
#define QP_DECL_F32(C, W)                                                                                      \
    extern template cudaError_t launch_pair<float, 1, C, kModeCsr, W>(const KArgs<float>&, int, cudaStream_t);  \
    extern template cudaError_t launch_pair<float, 2, C, kModeCsr, W>(const KArgs<float>&, int, cudaStream_t);  \
    extern template cudaError_t launch_pair<float, 1, C, kModeFull, W>(const KArgs<float>&, int, cudaStream_t); \
    extern template cudaError_t launch_pair<float, 2, C, kModeFull, W>(const KArgs<float>&, int, cudaStream_t);
#define QP_DECL_F64(C, MODE, W) \
    extern template cudaError_t launch_pair<double, 2, C, MODE, W>(const KArgs<double>&, int, cudaStream_t);
#define QP_DECL_F64_G1(C, MODE, W) \
    extern template cudaError_t launch_pair<double, 1, C, MODE, W>(const KArgs<double>&, int, cudaStream_t);
QP_DECL_F64_G1(2, kModeDist, 8) QP_DECL_F64_G1(4, kModeDist, 8) QP_DECL_F64_G1(8, kModeDist, 8)
QP_DECL_F32(2, 1) QP_DECL_F32(3, 1) QP_DECL_F32(4, 1) QP_DECL_F32(5, 1) QP_DECL_F32(6, 1) QP_DECL_F32(7, 1) QP_DECL_F32(8, 1)
QP_DECL_F32(9, 1) QP_DECL_F32(10, 1) QP_DECL_F32(11, 1) QP_DECL_F32(12, 1) QP_DECL_F32(13, 1) QP_DECL_F32(14, 1)
QP_DECL_F32(15, 1) QP_DECL_F32(16, 1) QP_DECL_F32(8, 4) QP_DECL_F32(12, 4) QP_DECL_F32(16, 4)
#define QP_DECL_F32_MB(C)                                                                                              \
    extern template cudaError_t launch_pair<float, 1, C, kModeCsr | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);  \
    extern template cudaError_t launch_pair<float, 2, C, kModeCsr | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);  \
    extern template cudaError_t launch_pair<float, 1, C, kModeFull | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t); \
    extern template cudaError_t launch_pair<float, 2, C, kModeFull | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);
QP_DECL_F32_MB(9) QP_DECL_F32_MB(10) QP_DECL_F32_MB(11) QP_DECL_F32_MB(12)
QP_DECL_F64(2, kModeFull, 1) QP_DECL_F64(4, kModeFull, 1) QP_DECL_F64(6, kModeFull, 1) QP_DECL_F64(8, kModeFull, 1)
QP_DECL_F64(8, kModeFull, 8) QP_DECL_F64(2, kModeDist, 8) QP_DECL_F64(4, kModeDist, 8) QP_DECL_F64(8, kModeDist, 8)

// ------------------------------------------------------------------------------------------------------------
// device-side scheduling kernels
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void set_status(SchedHeader* h, int code, int where) {
    if (atomicCAS(&h->status[0], 0, code) == 0) h->status[1] = where;
}

__global__ void k_check_residues(const uint8_t* __restrict__ seqs, const int64_t* __restrict__ offs, int k, int A,
                                 SchedHeader* h) {
    const int64_t lo = offs[0], hi = offs[k];
    for (int64_t q = lo + blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < hi; q += (int64_t)gridDim.x * blockDim.x)
        if (seqs[q] >= A) set_status(h, QP_ERR_BAD_RESIDUE, -1);
}

__global__ void k_classify(const int64_t* __restrict__ offs, int k, const int32_t* __restrict__ pairs, int64_t P,
                           uint32_t cmask, int fp64, int refine, PairInfo* __restrict__ info, int32_t* __restrict__ rows1,
                           int64_t* __restrict__ cells, SchedHeader* h) {
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= P) return;
    const int x = pairs[2 * p], y = pairs[2 * p + 1];
    PairInfo pi;
    pi.xoff = pi.yoff = 0;
    pi.n = pi.m = 0;
    pi.cls = -1;
    pi.nb = 0;
    pi.bin = 0;
    if (x < 0 || y < 0 || x >= k || y >= k || x == y) {
        set_status(h, QP_ERR_BAD_PAIR, (int)p);
    } else {
        const int64_t n = offs[x + 1] - offs[x], m = offs[y + 1] - offs[y];
        if (n < 1 || m < 1 || n > QP_MAX_LEN || m > QP_MAX_LEN) {
            set_status(h, QP_ERR_EMPTY_SEQUENCE, (int)p);
        } else {
            pi.xoff = offs[x];
            pi.yoff = offs[y];
            pi.n = (int)n;
            pi.m = (int)m;
            int nb;
            const int c = choose_class((int)n, (int)m + 1, cmask, fp64 != 0, &nb);   // never -1: the masks hold split classes
            pi.cls = (int16_t)c;
            pi.nb = (int16_t)nb;
            pi.bin = bin_of((uint64_t)slot_bytes((int)n, class_C(c, fp64 != 0), nb, fp64 ? 8 : 4));
            atomicAdd(&h->hist[c][pi.bin], 1u);
            if (refine) {   // the fp64 class the pair would be re-evaluated in, should it turn out near-identical
                int nbd;
                const int c64 = choose_class((int)n, (int)m + 1, kMaskRefine, true, &nbd);
                const unsigned long long sb = (unsigned long long)slot_bytes((int)n, class_C(c64, true), nbd, 8);
                if (h->rq.poll_slot_bytes[c64] < sb) atomicMax(&h->rq.poll_slot_bytes[c64], sb);
                if (h->rq.possible[c64] < kPollCtas) atomicAdd(&h->rq.possible[c64], 1);
            }
        }
    }
    info[p] = pi;
    rows1[p] = pi.n + 1;
    if (cells) cells[p] = (int64_t)pi.n * pi.m;
}

__global__ void k_bins(SchedHeader* h) {
    __shared__ int cnt[kNumClasses];
    const int c = threadIdx.x;
    if (c < kNumClasses) {
        uint32_t run = 0;
        for (int b = kNumBins - 1; b >= 0; --b) {
            h->bin_start[c][b] = run;
            run += h->hist[c][b];
        }
        cnt[c] = (int)run;
        h->cls_count[c] = (int)run;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int s = 0;
        for (int q = 0; q < kNumClasses; ++q) {
            h->cls_start[q] = s;
            s += cnt[q];
        }
    }
}

__global__ void k_scatter(const PairInfo* __restrict__ info, int64_t P, int32_t* __restrict__ order, SchedHeader* h) {
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= P) return;
    const int c = info[p].cls;
    if (c < 0) return;
    const int b = info[p].bin;
    const uint32_t pos = h->cls_start[c] + h->bin_start[c][b] + atomicAdd(&h->bin_fill[c][b], 1u);
    order[pos] = (int32_t)p;
}

struct MaxW {
    int w[kNumClasses];
};

// grant resident warps per class under the slot budget, then lay the slots out
__global__ void k_slots(const PairInfo* __restrict__ info, const int32_t* __restrict__ order, MaxW maxw,
                        int64_t avail, int64_t* __restrict__ slot_off, SchedHeader* h) {
    __shared__ int64_t sh[1024];
    __shared__ int W[kNumClasses], W0[kNumClasses + 1];
    __shared__ int done, fail;
    const int t = threadIdx.x;
    const int64_t early = (int64_t)h->poll_bytes;   // head of the slot region: slots of the fp64 pollers
    avail -= early;
    for (int shift = 0;; ++shift) {
        if (t == 0) {
            int s = 0, all1 = 1;
            for (int c = 0; c < kNumClasses; ++c) {
                int cnt = h->cls_count[c];
                int w = cnt ? max(1, min(cnt, maxw.w[c] >> shift)) : 0;
                if (w > 1) all1 = 0;
                W[c] = w;
                W0[c] = s;
                s += w;
            }
            W0[kNumClasses] = s;
            done = all1;
        }
        __syncthreads();
        const int N = W0[kNumClasses];
        const int per = (N + blockDim.x - 1) / blockDim.x;
        int64_t loc = 0;
        for (int q = t * per; q < min(N, (t + 1) * per); ++q) {
            int c = 0;
            while (q >= W0[c + 1]) ++c;
            loc += (int64_t)bin_ub(info[order[h->cls_start[c] + (q - W0[c])]].bin);
        }
        int64_t tot;
        int64_t ex = block_excl_scan(loc, sh, &tot);
        if (tot <= avail) {
            for (int q = t * per; q < min(N, (t + 1) * per); ++q) {
                int c = 0;
                while (q >= W0[c + 1]) ++c;
                slot_off[q] = early + ex;
                ex += (int64_t)bin_ub(info[order[h->cls_start[c] + (q - W0[c])]].bin);
            }
            if (t == 0) fail = 0;
            break;
        }
        if (done) {
            if (t == 0) fail = 1;
            break;
        }
        __syncthreads();
    }
    __syncthreads();
    if (t < kNumClasses) {
        h->cls_W[t] = fail ? 0 : W[t];
        h->cls_slot0[t] = W0[t];
        h->cls_cursor[t] = W[t];
    }
    if (t == 0 && fail) set_status(h, QP_ERR_WORKSPACE_TOO_SMALL, -1);
}

__global__ void k_copy_pool(const int32_t* __restrict__ nnz, const int64_t* __restrict__ pool_off,
                            const int64_t* __restrict__ base, int64_t P, const float2* __restrict__ pool,
                            int64_t cap, int32_t* __restrict__ col,
                            float* __restrict__ val) {
    const int64_t p = blockIdx.x * (int64_t)(blockDim.x >> 5) + (threadIdx.x >> 5);
    if (p >= P) return;
    const int lane = threadIdx.x & 31;
    const int64_t cnt = nnz[p], src = pool_off[p], dst = base[p];
    if (src + cnt > cap || dst + cnt > cap) return;
    for (int64_t q = lane; q < cnt; q += 32) {
        const float2 e = pool[src + q];
        col[dst + q] = __float_as_int(e.y);
        val[dst + q] = e.x;
    }
}

struct MaxW64 {
    int w[kNumClasses];
};
// Slot plan of the fp64 re-evaluation queue (RefineQ in qp_internal.h).
// which = 0, schedule time, before k_slots: the pollers' slots come off the head of the slot region, at most half of
//   it: up to poll_max (poll_ctas(sms)) slots per class that can receive pairs, each sized for the largest pair of the class; classes
//   are served in ascending slot size and a class that does not fit gets fewer pollers or none (the drainers take
//   its pairs). What was taken is recorded in poll_bytes; the fp32 slots start behind it.
// which = 1, after the fp32 classes have joined: the drainers' slots reuse the fp32 slot region; one slot for every
//   class with pairs left (a misfit is an error), then the rest of the region class by class.
__global__ void k_refine_plan(int which, MaxW64 maxw, int poll_max, int64_t avail, const PairInfo* __restrict__ info,
                              const int32_t* __restrict__ order, SchedHeader* h) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    RefineQ& rq = h->rq;
    if (which == 0) {
        // the pollers never take what the fp32 classes need at the least (one slot per class, sized for its largest
        // pair -- the first of its list): a workspace of exactly the minimum that qp_workspace_bytes reports must do
        long long fp32_min = 0;
        for (int c = 0; c < kNumClasses; ++c)
            if (h->cls_count[c] > 0) fp32_min += (long long)bin_ub(info[order[h->cls_start[c]]].bin);
        const long long spare = (long long)avail - fp32_min;
        unsigned long long room = (unsigned long long)min((long long)avail / 2, max(spare, 0ll)), used = 0;
        for (int c = kNumPacked; c < kSplitEnd; ++c) {   // slot sizes grow with the class index
            const unsigned long long sb = (rq.poll_slot_bytes[c] + 255ull) & ~255ull;
            rq.poll_slot_bytes[c] = sb;
            int W = 0;
            if (rq.possible[c] > 0 && sb > 0) W = (int)min((long long)min(rq.possible[c], poll_max), (long long)((room - used) / sb));
            rq.Wpoll[c] = W;
            rq.poll_slot0[c] = used;
            used += (unsigned long long)W * sb;
        }
        h->poll_bytes = used;
        return;
    }
    const unsigned long long lo = h->poll_bytes, bytes = (unsigned long long)avail - lo;
    unsigned long long base = 0;
    int left[kNumClasses];
    for (int c = 0; c < kNumClasses; ++c) {
        rq.slot_bytes[c] = (rq.slot_bytes[c] + 255ull) & ~255ull;
        left[c] = max(0, rq.count[c] - min(rq.cursor[c], rq.count[c]));   // the pollers are still pulling: an upper bound
        if (left[c] > 0) base += rq.slot_bytes[c];
    }
    const bool fits = base <= bytes;
    if (!fits) set_status(h, QP_ERR_WORKSPACE_TOO_SMALL, -1);
    unsigned long long spare = fits ? bytes - base : 0, used = 0;
    for (int c = 0; c < kNumClasses; ++c) {
        int W = 0;
        if (left[c] > 0 && fits) {
            const unsigned long long sb = rq.slot_bytes[c];
            const long long extra = min((long long)min(left[c], maxw.w[c]) - 1, (long long)(spare / sb));
            W = 1 + (int)max(extra, 0ll);
            spare -= (unsigned long long)(W - 1) * sb;
            rq.slot0[c] = lo + used;
            used += (unsigned long long)W * sb;
        }
        rq.W[c] = W;
    }
}

__global__ void k_finish(const SchedHeader* h, int32_t* status) {
    if (threadIdx.x < 3) status[threadIdx.x] = h->status[threadIdx.x];
    if (threadIdx.x == 3) {   // pairs whose distance was re-evaluated in fp64
        int t = 0;
        for (int c = 0; c < kNumClasses; ++c) t += h->rq.count[c];
        status[3] = t;
    }
}

// ------------------------------------------------------------------------------------------------------------
// host
// ------------------------------------------------------------------------------------------------------------
static thread_local int g_launches = 0;
static thread_local int g_profile = 0;
static thread_local bool g_want_hist = false;                      // set by qp_posteriors_budgeted around its passes
static thread_local unsigned long long g_tau_hist[kTauBins];      // host copy of the last budgeted call's histogram
static thread_local float g_tau0 = 0.f;
static thread_local bool g_tau_hist_valid = false;

// Per host thread and device: side streams so that the per-class kernels overlap their tails, the events that fork
// and join them, and the profiling events. Created on the first call on a device, kept until qp_shutdown().
constexpr int kNumRefine = kSplitEnd - kNumPacked;            // split fp64 classes of the re-evaluation queues
constexpr int kNumStreams = kNumClasses + kNumRefine + 1;     // fp32 / QP_FP64 classes | early fp64 queue | CSR placement
struct Ctx {
    bool ok = false;
    int dev = -1, sms = kSmAssumed;
    cudaStream_t st[kNumStreams];
    cudaEvent_t fork, fork2, join[kNumStreams];
    cudaEvent_t pev[5];                  // phase boundaries on the caller's stream
    cudaEvent_t cev[2 * kNumClasses];    // per class: start / stop on its side stream
    bool prof_valid = false;
};
constexpr int kMaxDevices = 64;
static thread_local Ctx* g_ctxs[kMaxDevices] = {nullptr};
static thread_local Ctx* g_ctx = nullptr;     // context of the last call on this thread

static void ctx_destroy(Ctx* c) {
    if (!c) return;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) {   // no usable runtime (e.g. process teardown): only the host object goes
        (void)cudaGetLastError();
        delete c;
        return;
    }
    if (c->dev >= 0) cudaSetDevice(c->dev);
    if (c->ok) {
        for (int q = 0; q < kNumStreams; ++q) {
            cudaStreamDestroy(c->st[q]);
            cudaEventDestroy(c->join[q]);
        }
        cudaEventDestroy(c->fork);
        cudaEventDestroy(c->fork2);
        for (int q = 0; q < 5; ++q) cudaEventDestroy(c->pev[q]);
        for (int q = 0; q < 2 * kNumClasses; ++q) cudaEventDestroy(c->cev[q]);
    }
    if (cur >= 0) cudaSetDevice(cur);
    (void)cudaGetLastError();
    delete c;
}

// A host thread that exits without qp_shutdown() must not leak its 26 streams and ~75 events per device: the first
// context a thread creates arms this owner, whose destructor runs at thread exit and releases what is left.
struct CtxOwner {
    bool armed = false;
    ~CtxOwner() {
        if (!armed) return;
        for (int d = 0; d < kMaxDevices; ++d) {
            ctx_destroy(g_ctxs[d]);
            g_ctxs[d] = nullptr;
        }
        g_ctx = nullptr;
    }
};
static thread_local CtxOwner g_ctx_owner;

static Ctx* ctx_get() {
    int dev;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
    if (g_ctxs[dev] && g_ctxs[dev]->ok) return g_ctx = g_ctxs[dev];
    Ctx* c = new Ctx();
    c->dev = dev;
    bool ok = cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess;
    for (int q = 0; q < kNumStreams && ok; ++q)
        ok = cudaStreamCreateWithFlags(&c->st[q], cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&c->join[q], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&c->fork, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->fork2, cudaEventDisableTiming) == cudaSuccess;
    for (int q = 0; q < 5 && ok; ++q) ok = cudaEventCreate(&c->pev[q]) == cudaSuccess;
    for (int q = 0; q < 2 * kNumClasses && ok; ++q) ok = cudaEventCreate(&c->cev[q]) == cudaSuccess;
    if (!ok) {   // partial creation: nothing is kept
        (void)cudaGetLastError();
        delete c;
        return nullptr;
    }
    c->ok = true;
    g_ctxs[dev] = c;
    g_ctx_owner.armed = true;
    return g_ctx = c;
}

static void prof_class(Ctx* c, int cls, int which, cudaStream_t st) {
    if (g_profile) cudaEventRecord(c->cev[2 * cls + which], st);
}
static void prof_mark(Ctx* c, int i, cudaStream_t st) {
    if (!g_profile) return;
    cudaEventRecord(c->pev[i], st);
    if (i == 4) c->prof_valid = true;
}

static inline int64_t align256(int64_t v) { return (v + 255) & ~(int64_t)255; }

struct Layout {   // byte offsets inside the workspace
    int64_t hdr, info, order, rows1, cells, nnz, pool_off, dense_off, slot_off, refine_list, tau_hist, scan_tmp, pool, slots;
    int64_t fixed;   // everything before the slots
};

static Layout make_layout(int64_t P, int64_t nnz_cap, bool dense, int64_t max_slots) {
    Layout L;
    int64_t o = 0;
    auto take = [&](int64_t bytes) {
        int64_t r = o;
        o += align256(bytes);
        return r;
    };
    L.hdr = take(sizeof(SchedHeader));
    L.info = take(P * (int64_t)sizeof(PairInfo));
    L.order = take(P * 4);
    L.rows1 = take(P * 4);
    L.cells = take(dense ? P * 8 : 0);
    L.nnz = take(P * 4);
    L.pool_off = take(P * 8);
    L.dense_off = take(dense ? (P + 1) * 8 : 0);
    L.slot_off = take(max_slots * 8);
    L.refine_list = take((int64_t)kNumRefine * (P + kListPad) * 4);
    L.tau_hist = take((int64_t)kTauBins * 8);
    L.scan_tmp = take((P / kScanChunk + 2) * 2 * 8);
    L.pool = take(nnz_cap * 8);
    L.slots = o;
    L.fixed = o;
    return L;
}

// scratch slots (= pairs in flight) a class can use: one per warp (packed) or per CTA (split)
static int max_units(int cls, bool fp64, int sms) {
    const int C = class_C(cls, fp64), W = class_W(cls, fp64);
    return C == 0 ? 0 : sms * ctas_per_sm(C, W, fp64) * units_per_cta(W);
}
static int class_grid(int cls, bool fp64, int sms) { return sms * ctas_per_sm(class_C(cls, fp64), class_W(cls, fp64), fp64); }
static int64_t total_max_slots(int sms) {
    int64_t s = 0;
    for (int c = 0; c < kNumClasses; ++c) s += std::max(max_units(c, false, sms), max_units(c, true, sms));
    return s;
}

static int check_model(const qp_model& m) {
    if (m.n_ins < 1 || m.n_ins > QP_MAX_INS) return QP_ERR_INVALID_ARG;
    if (m.alphabet < 2 || m.alphabet > QP_MAX_ALPHABET) return QP_ERR_INVALID_ARG;
    if (!m.log_match || !m.log_ins) return QP_ERR_INVALID_ARG;
    return QP_OK;
}
static int check_params(const qp_params* p) {
    if (!p) return QP_ERR_INVALID_ARG;
    int r = check_model(p->hmm);
    if (r) return r;
    r = check_model(p->pf);
    if (r) return r;
    if (p->hmm.alphabet != p->pf.alphabet) return QP_ERR_INVALID_ARG;
    if (!(p->threshold > 0.0) || !(p->threshold <= 1.0)) return QP_ERR_INVALID_ARG;
    if (p->precision != QP_FP32 && p->precision != QP_FP64) return QP_ERR_INVALID_ARG;
    return QP_OK;
}

// linear-space weights after the background normalisation (posterior-invariant, SURVEY.md 8(c) pin 8):
// em(a,b) = exp(lm[a][b] - lx[a] - lx[b]), insert emissions 1. Returns log2 of the largest per-row growth.
template <typename R> static double prep_model(const qp_model& m, Weights<R>& w, double* em /*32x32*/, double* lx) {
    const int A = m.alphabet;
    auto ex = [](double v) { return v == -INFINITY ? 0.0 : std::exp(v); };
    double emax = 0.0;
    for (int a = 0; a < kTabDim; ++a) {
        lx[a] = a < A ? m.log_ins[a] : 0.0;
        for (int b = 0; b < kTabDim; ++b) {
            double v = 0.0;
            if (a < A && b < A) v = ex(m.log_match[a * A + b] - m.log_ins[a] - m.log_ins[b]);
            em[a * kTabDim + b] = v;
            emax = std::max(emax, v);
        }
    }
    w.wMM = (R)ex(m.t_MM);
    w.initM = (R)ex(m.init_M);
    w.endM = (R)ex(m.end_M);
    double wsum = ex(m.t_MM);
    for (int g = 0; g < kMaxIns; ++g) {
        const bool on = g < m.n_ins;
        w.wMI[g] = on ? (R)ex(m.t_MI[g]) : R(0);
        w.wII[g] = on ? (R)ex(m.t_II[g]) : R(0);
        w.wIM[g] = on ? (R)ex(m.t_IM[g]) : R(0);
        w.initI[g] = on ? (R)ex(m.init_I[g]) : R(0);
        w.endI[g] = on ? (R)ex(m.end_I[g]) : R(0);
        if (on) wsum += 2.0 * ex(m.t_IM[g]) + ex(m.t_II[g]) + ex(m.t_MI[g]);
    }
    return std::log2(std::max(1.0, emax) * std::max(1.0, wsum));
}

template <typename R> static int fill_kargs(const qp_params* prm, KArgs<R>& ka) {
    double eh[kTabDim * kTabDim], ep[kTabDim * kTabDim];
    const double gh = prep_model<R>(prm->hmm, ka.wh, eh, ka.lx_h);
    const double gp = prep_model<R>(prm->pf, ka.wp, ep, ka.lx_p);
    for (int q = 0; q < kTabDim * kTabDim; ++q) {
        ka.tab[q].x = (R)eh[q];
        ka.tab[q].y = (R)ep[q];
        if (!std::isfinite((double)ka.tab[q].x) || !std::isfinite((double)ka.tab[q].y)) return QP_ERR_RANGE;
    }
    // renormalise often enough that values cannot leave the exponent range between two renormalisations
    const double g = std::max(gh, gp), room = sizeof(R) == 4 ? 56.0 : 500.0;
    int every = 8;
    while (every > 1 && every * g > room) every >>= 1;
    if (every * g > room) return QP_ERR_RANGE;
    ka.rescale_mask = every - 1;
    ka.tau = (R)prm->threshold;
    if constexpr (sizeof(R) == 4) ka.w2.set(ka.wh, ka.wp);
    return QP_OK;
}

static int launch_class_f32(int gp, bool full, int cls, const KArgs<float>& ka, int grid, cudaStream_t st) {
    cudaError_t e = cudaErrorInvalidValue;
#define QP_CASE(CLS, C, W)                                                                                          \
    case CLS:                                                                                                       \
        if (full) e = gp == 1 ? launch_pair<float, 1, C, kModeFull, W>(ka, grid, st) : launch_pair<float, 2, C, kModeFull, W>(ka, grid, st); \
        else e = gp == 1 ? launch_pair<float, 1, C, kModeCsr, W>(ka, grid, st) : launch_pair<float, 2, C, kModeCsr, W>(ka, grid, st);        \
        break;
    switch (cls) {
        QP_CASE(0, 2, 1) QP_CASE(1, 3, 1) QP_CASE(2, 4, 1) QP_CASE(3, 5, 1) QP_CASE(4, 6, 1) QP_CASE(5, 7, 1)
        QP_CASE(6, 8, 1) QP_CASE(7, 9, 1) QP_CASE(8, 10, 1) QP_CASE(9, 11, 1) QP_CASE(10, 12, 1) QP_CASE(11, 13, 1)
        QP_CASE(12, 14, 1) QP_CASE(13, 15, 1) QP_CASE(14, 16, 1) QP_CASE(15, 8, 4) QP_CASE(16, 12, 4) QP_CASE(17, 16, 4)
#define QP_CASE_MB(CLS, C)                                                                                          \
    case CLS:                                                                                                       \
        if (full) e = gp == 1 ? launch_pair<float, 1, C, kModeFull | kModeMB, 1>(ka, grid, st) : launch_pair<float, 2, C, kModeFull | kModeMB, 1>(ka, grid, st); \
        else e = gp == 1 ? launch_pair<float, 1, C, kModeCsr | kModeMB, 1>(ka, grid, st) : launch_pair<float, 2, C, kModeCsr | kModeMB, 1>(ka, grid, st);        \
        break;
        QP_CASE_MB(18, 9) QP_CASE_MB(19, 10) QP_CASE_MB(20, 11) QP_CASE_MB(21, 12)
#undef QP_CASE_MB
    }
#undef QP_CASE
    ++g_launches;
    return e == cudaSuccess ? QP_OK : QP_ERR_CUDA;
}
static int launch_class_f64(bool dist_only, int gp, int cls, const KArgs<double>& ka, int grid, cudaStream_t st) {
    cudaError_t e = cudaErrorInvalidValue;
    if (!dist_only) {
        switch (cls) {
            case 0: e = launch_pair<double, 2, 2, kModeFull, 1>(ka, grid, st); break;
            case 2: e = launch_pair<double, 2, 4, kModeFull, 1>(ka, grid, st); break;
            case 4: e = launch_pair<double, 2, 6, kModeFull, 1>(ka, grid, st); break;
            case 6: e = launch_pair<double, 2, 8, kModeFull, 1>(ka, grid, st); break;
            case 17: e = launch_pair<double, 2, 8, kModeFull, 8>(ka, grid, st); break;
        }
    } else {
        switch (cls) {
            // the distance-only kernels exist for one and for two insert-state pairs in the partition function
            case 15: e = gp == 1 ? launch_pair<double, 1, 2, kModeDist, 8>(ka, grid, st) : launch_pair<double, 2, 2, kModeDist, 8>(ka, grid, st); break;
            case 16: e = gp == 1 ? launch_pair<double, 1, 4, kModeDist, 8>(ka, grid, st) : launch_pair<double, 2, 4, kModeDist, 8>(ka, grid, st); break;
            case 17: e = gp == 1 ? launch_pair<double, 1, 8, kModeDist, 8>(ka, grid, st) : launch_pair<double, 2, 8, kModeDist, 8>(ka, grid, st); break;
        }
    }
    ++g_launches;
    return e == cudaSuccess ? QP_OK : QP_ERR_CUDA;
}

template <typename R> static void fill_common(KArgs<R>& ka, const uint8_t* d_seqs, const int32_t* d_pairs, int32_t k,
                                              char* ws, const Layout& L, const qp_output* out, int64_t P) {
    ka.k = k;
    ka.seqs = d_seqs;
    ka.pairs = d_pairs;
    ka.info = (const PairInfo*)(ws + L.info);
    ka.order = (const int32_t*)(ws + L.order);
    ka.hdr = (SchedHeader*)(ws + L.hdr);
    ka.slot_off = (const int64_t*)(ws + L.slot_off);
    ka.slots = ws + L.slots;
    ka.refine_list = (int32_t*)(ws + L.refine_list);
    ka.refine_stride = P + kListPad;
    ka.producers_total = 0;
    ka.tau_hist = nullptr;
    ka.tau_bits0 = 0;
    ka.refine_cmask = kMaskRefine;
    ka.pair_row_base = out->pair_row_base;
    ka.row_ptr = out->row_ptr;
    ka.pool = (float2*)(ws + L.pool);
    ka.pool_cap = out->nnz_capacity;
    ka.nnz = (int32_t*)(ws + L.nnz);
    ka.pool_off = (int64_t*)(ws + L.pool_off);
    ka.dist = out->dist;
    ka.dense_P = out->dense_P;
    ka.dense_off = (const int64_t*)(ws + L.dense_off);
    ka.logZ = out->logZ;
}

#define QP_CUDA(x)                                  \
    do {                                            \
        if ((x) != cudaSuccess) return QP_ERR_CUDA; \
    } while (0)

}  // namespace qp

using namespace qp;

extern "C" int qp_last_launch_count(void) { return g_launches; }

extern "C" void qp_set_profile(int on) {
    g_profile = on;
    if (!on && g_ctx) g_ctx->prof_valid = false;
}

extern "C" int qp_get_profile_classes(float start_ms[QP_NUM_CLASSES], float stop_ms[QP_NUM_CLASSES]) {
    static_assert(QP_NUM_CLASSES == kNumClasses, "qp.h and qp_internal.h disagree");
    if (!g_ctx || !g_ctx->prof_valid || !start_ms || !stop_ms) return QP_ERR_INVALID_ARG;
    for (int c = 0; c < kNumClasses; ++c) {
        start_ms[c] = stop_ms[c] = -1.0f;
        if (cudaEventQuery(g_ctx->cev[2 * c]) != cudaSuccess) { (void)cudaGetLastError(); continue; }
        if (cudaEventElapsedTime(&start_ms[c], g_ctx->pev[1], g_ctx->cev[2 * c]) != cudaSuccess ||
            cudaEventElapsedTime(&stop_ms[c], g_ctx->pev[1], g_ctx->cev[2 * c + 1]) != cudaSuccess) {
            (void)cudaGetLastError();
            start_ms[c] = stop_ms[c] = -1.0f;
        }
    }
    return QP_OK;
}

extern "C" int qp_get_profile(float ms[4]) {
    if (!g_ctx || !g_ctx->prof_valid || !ms) return QP_ERR_INVALID_ARG;
    for (int q = 0; q < 4; ++q)
        if (cudaEventElapsedTime(&ms[q], g_ctx->pev[q], g_ctx->pev[q + 1]) != cudaSuccess) return QP_ERR_CUDA;
    return QP_OK;
}

extern "C" void qp_shutdown(void) {
    for (int d = 0; d < kMaxDevices; ++d) {
        ctx_destroy(g_ctxs[d]);
        g_ctxs[d] = nullptr;
    }
    g_ctx = nullptr;
}

extern "C" const char* qp_version(void) { return "qp-b200 0.2 (sm_100a)"; }

extern "C" const char* qp_status_string(int s) {
    switch (s) {
        case QP_OK: return "ok";
        case QP_ERR_INVALID_ARG: return "invalid argument";
        case QP_ERR_BAD_RESIDUE: return "residue code >= alphabet";
        case QP_ERR_EMPTY_SEQUENCE: return "empty or over-long sequence";
        case QP_ERR_BAD_PAIR: return "pair index out of range or x == y";
        case QP_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case QP_ERR_NNZ_CAPACITY: return "nnz capacity exceeded";
        case QP_ERR_CUDA: return "CUDA runtime error";
        case QP_ERR_RANGE: return "model weights outside the supported dynamic range";
        case QP_ERR_STATIC_LIMIT: return "more sequences than the built-in scratch of qp_guide_tree_static holds (1024)";
        default: return "unknown status";
    }
}

extern "C" int qp_workspace_bytes(const int64_t* h_offsets, int32_t k, const int32_t* h_pairs, int64_t P,
                                  const qp_params* params, int64_t nnz_capacity, int want_dense, size_t budget_bytes,
                                  size_t* out_bytes) {
    if (!h_offsets || (!h_pairs && P > 0) || !out_bytes || k < 0 || P < 0 || nnz_capacity < 0) return QP_ERR_INVALID_ARG;
    int r = check_params(params);
    if (r) return r;
    const bool fp64 = params->precision == QP_FP64;
    const uint32_t cmask = fp64 ? kMaskF64 : kMaskF32;
    const int rb = fp64 ? 8 : 4;
    const bool refine = !fp64 && !(params->flags & QP_FLAG_NO_REFINE);
    int sms = kSmAssumed;
    {
        int dev;
        if (cudaGetDevice(&dev) == cudaSuccess) {
            int v;
            if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sms = v;
        } else {
            (void)cudaGetLastError();
        }
    }
    const Layout L = make_layout(P, nnz_capacity, want_dense != 0, total_max_slots(sms));
    std::vector<std::vector<uint64_t>> sz(kNumClasses);
    uint64_t sz64[kNumClasses] = {0};   // largest fp64 slot per class among the pairs a refinement pass could see
    int64_t cnt64[kNumClasses] = {0};   // ... and how many pairs the class could receive
    for (int64_t p = 0; p < P; ++p) {
        const int x = h_pairs[2 * p], y = h_pairs[2 * p + 1];
        if (x < 0 || y < 0 || x >= k || y >= k || x == y) return QP_ERR_BAD_PAIR;
        const int64_t n = h_offsets[x + 1] - h_offsets[x], m = h_offsets[y + 1] - h_offsets[y];
        if (n < 1 || m < 1 || n > QP_MAX_LEN || m > QP_MAX_LEN) return QP_ERR_EMPTY_SEQUENCE;
        int nb;
        const int c = choose_class((int)n, (int)m + 1, cmask, fp64, &nb);
        sz[c].push_back(bin_ub(bin_of((uint64_t)slot_bytes((int)n, class_C(c, fp64), nb, rb))));
        if (refine) {
            const int c2 = choose_class((int)n, (int)m + 1, kMaskRefine, true, &nb);
            sz64[c2] = std::max(sz64[c2], (uint64_t)slot_bytes((int)n, class_C(c2, true), nb, 8));
            ++cnt64[c2];
        }
    }
    uint64_t full = 0, minimum = 0;
    for (int c = 0; c < kNumClasses; ++c) {
        std::sort(sz[c].begin(), sz[c].end(), std::greater<uint64_t>());
        const size_t W = std::min<size_t>(sz[c].size(), (size_t)max_units(c, fp64, sms));
        for (size_t w = 0; w < W; ++w) full += sz[c][w];
        if (!sz[c].empty()) minimum += sz[c][0];
    }
    // the drainers of the fp64 re-evaluation queue reuse the fp32 slots: every fp64 class must fit its largest slot once
    uint64_t ref_min = 0;
    for (uint64_t v : sz64) ref_min += v;
    minimum = std::max(minimum, ref_min);
    // ... and, budget permitting, once per resident CTA (capped at 4 GiB: which pairs get re-evaluated is only known
    // on the device)
    uint64_t ref_full = 0;
    for (int c = 0; c < kNumClasses; ++c)
        if ((kMaskRefine >> c) & 1) ref_full += sz64[c] * (uint64_t)std::min<int64_t>(cnt64[c], max_units(c, true, sms));
    full = std::max(full, std::min<uint64_t>(ref_full, 4ull << 30));
    // the pollers run beside the fp32 classes in a region of their own (at most half of the slot region, k_refine_plan):
    // at most kPollCtas slots per class that can receive pairs (this query does not touch the device: the upper bound)
    uint64_t poll_full = 0;
    for (int c = 0; c < kNumClasses; ++c)
        if ((kMaskRefine >> c) & 1) poll_full += sz64[c] * (uint64_t)std::min<int64_t>(cnt64[c], kPollCtas);
    full = std::max(std::max(full + poll_full, 2 * poll_full), minimum);
    const uint64_t need_min = (uint64_t)L.fixed + minimum, need_full = (uint64_t)L.fixed + full;
    if (budget_bytes != 0 && budget_bytes < need_min) {
        *out_bytes = (size_t)need_min;
        return QP_ERR_WORKSPACE_TOO_SMALL;
    }
    *out_bytes = (size_t)((budget_bytes != 0 && budget_bytes < need_full) ? budget_bytes : need_full);
    return QP_OK;
}

// the work of qp_posteriors after argument validation; every error after the first enqueue goes through `fail`,
// which waits for the side streams so that nothing is still writing the caller's buffers when the call returns
static int run_posteriors(Ctx* cx, const uint8_t* d_seqs, const int64_t* d_offsets, int32_t k, const int32_t* d_pairs,
                          int64_t P, const qp_params* params, void* d_workspace, size_t workspace_bytes,
                          const qp_output* out, cudaStream_t st) {
    const bool fp64 = params->precision == QP_FP64;
    const bool dense = out->dense_P != nullptr;
    const int sms = cx->sms;
    const bool refine = !fp64 && !(params->flags & QP_FLAG_NO_REFINE);
    const bool pollers = refine && !(params->flags & QP_FLAG_NO_POLLERS);
    const bool full_outputs = out->dense_P != nullptr || out->logZ != nullptr;   // test outputs: separate kernel instances
    const Layout L = make_layout(P, out->nnz_capacity, dense, total_max_slots(sms));
    if ((int64_t)workspace_bytes < L.fixed + 256) return QP_ERR_WORKSPACE_TOO_SMALL;
    char* ws = (char*)d_workspace;
    SchedHeader* hdr = (SchedHeader*)(ws + L.hdr);
    const int64_t avail = (int64_t)workspace_bytes - L.slots;

    // ---- host-side preparation of the kernel arguments (can fail: before anything is enqueued) ----------------
    std::vector<char> buf32(sizeof(KArgs<float>)), buf64(sizeof(KArgs<double>));
    KArgs<float>* ka32 = new (buf32.data()) KArgs<float>();
    KArgs<double>* ka64 = new (buf64.data()) KArgs<double>();
    int r;
    if (!fp64) {
        r = fill_kargs<float>(params, *ka32);
        if (r) return r;
        fill_common(*ka32, d_seqs, d_pairs, k, ws, L, out, P);
        ka32->refine_pass = 0;
        ka32->refine_below = refine ? (float)(params->refine_below > 0.0 ? params->refine_below : 0.25) : -1.0f;
    }
    if (fp64 || refine) {
        r = fill_kargs<double>(params, *ka64);
        if (r) return r;
        fill_common(*ka64, d_seqs, d_pairs, k, ws, L, out, P);
        ka64->refine_pass = 0;
        ka64->refine_below = -1.0f;
    }

    if (g_want_hist) {   // memory-limited mode: histogram of the kept values over threshold bins (qp_posteriors_budgeted)
        float t0 = (float)params->threshold;
        int32_t bits;
        memcpy(&bits, &t0, 4);
        ka32->tau_hist = ka64->tau_hist = (unsigned long long*)(ws + L.tau_hist);
        ka32->tau_bits0 = ka64->tau_bits0 = bits;
    }
    bool forked = false;
    auto fail = [&](int code) {
        if (forked)
            for (int q = 0; q < kNumStreams; ++q) cudaStreamSynchronize(cx->st[q]);
        (void)cudaGetLastError();
        return code;
    };
#define QP_TRY(x)                                          \
    do {                                                   \
        if ((x) != cudaSuccess) return fail(QP_ERR_CUDA);  \
    } while (0)

    QP_TRY(cudaMemsetAsync(hdr, 0, sizeof(SchedHeader), st));
    prof_mark(cx, 0, st);
    QP_TRY(cudaMemsetAsync(ws + L.nnz, 0, (size_t)P * 4, st));
    if (refine) QP_TRY(cudaMemsetAsync(ws + L.refine_list, 0xff, (size_t)kNumRefine * (P + kListPad) * 4, st));   // -1 = empty
    if (g_want_hist) QP_TRY(cudaMemsetAsync(ws + L.tau_hist, 0, (size_t)kTauBins * 8, st));

    // ---- a0: schedule, entirely on the device --------------------------------------------------------------
    const uint32_t cmask = fp64 ? kMaskF64 : kMaskF32;
    const int pb = (int)((P + 255) / 256);
    k_check_residues<<<2 * sms, 256, 0, st>>>(d_seqs, d_offsets, k, params->hmm.alphabet, hdr);
    k_classify<<<pb, 256, 0, st>>>(d_offsets, k, d_pairs, P, cmask, fp64 ? 1 : 0, refine ? 1 : 0, (PairInfo*)(ws + L.info),
                                   (int32_t*)(ws + L.rows1), dense ? (int64_t*)(ws + L.cells) : nullptr, hdr);
    k_bins<<<1, 32, 0, st>>>(hdr);
    k_scatter<<<pb, 256, 0, st>>>((const PairInfo*)(ws + L.info), P, (int32_t*)(ws + L.order), hdr);
    g_launches += 4;
    MaxW64 mw64;
    for (int c = 0; c < kNumClasses; ++c) mw64.w[c] = ((kMaskRefine >> c) & 1) ? max_units(c, true, sms) : 0;
    if (pollers) {   // the pollers' slots come off the head of the slot region
        k_refine_plan<<<1, 32, 0, st>>>(0, mw64, poll_ctas(sms), avail, (const PairInfo*)(ws + L.info), (const int32_t*)(ws + L.order), hdr);
        ++g_launches;
    }
    MaxW mw;
    for (int c = 0; c < kNumClasses; ++c) mw.w[c] = ((cmask >> c) & 1) ? max_units(c, fp64, sms) : 0;
    k_slots<<<1, 1024, 0, st>>>((const PairInfo*)(ws + L.info), (const int32_t*)(ws + L.order), mw, avail,
                                (int64_t*)(ws + L.slot_off), hdr);
    ++g_launches;
    scan_launch<int32_t>((const int32_t*)(ws + L.rows1), P, out->pair_row_base, (int64_t*)(ws + L.scan_tmp), st, &g_launches);
    if (dense) scan_launch<int64_t>((const int64_t*)(ws + L.cells), P, (int64_t*)(ws + L.dense_off), (int64_t*)(ws + L.scan_tmp), st, &g_launches);
    QP_TRY(cudaGetLastError());

    // ---- a1..a7: one persistent kernel per class, forked onto side streams ----------------------------------
    if (pollers) {   // pollers leave when this many fp32 class warps have exited
        int total = 0;
        for (int c = 0; c < kNumClasses; ++c)
            if ((cmask >> c) & 1) total += class_grid(c, false, sms) * (class_W(c, false) == 1 ? kWarpsPerCta : class_W(c, false));
        ka32->producers_total = ka64->producers_total = total;
    }
    prof_mark(cx, 1, st);
    QP_TRY(cudaEventRecord(cx->fork, st));
    forked = true;
    // launch order: the split classes (the longest pairs: they set the tail) first, then the two-block classes, then
    // the one-block classes from wide to narrow
    int launch_order[kNumClasses], nl = 0;
    for (int c = kSplitEnd - 1; c >= kNumPacked; --c) launch_order[nl++] = c;
    for (int c = kNumClasses - 1; c >= kSplitEnd; --c) launch_order[nl++] = c;
    for (int c = kNumPacked - 1; c >= 0; --c) launch_order[nl++] = c;
    for (int q = 0; q < nl; ++q) {
        const int c = launch_order[q];
        if (!((cmask >> c) & 1)) continue;
        QP_TRY(cudaStreamWaitEvent(cx->st[c], cx->fork, 0));
        const int grid = class_grid(c, fp64, sms);
        prof_class(cx, c, 0, cx->st[c]);
        r = fp64 ? launch_class_f64(false, 2, c, *ka64, grid, cx->st[c])
                 : launch_class_f32(params->pf.n_ins, full_outputs, c, *ka32, grid, cx->st[c]);
        if (r) return fail(r);
        prof_class(cx, c, 1, cx->st[c]);
        QP_TRY(cudaEventRecord(cx->join[c], cx->st[c]));
        QP_TRY(cudaStreamWaitEvent(st, cx->join[c], 0));
    }
    if (pollers) {   // pollers of the fp64 re-evaluation queue, behind the fp32 classes: they fill the room those leave
        ka64->refine_pass = 1;
        for (int c = kSplitEnd - 1; c >= kNumPacked; --c) {
            cudaStream_t es = cx->st[kNumClasses + (c - kNumPacked)];
            QP_TRY(cudaStreamWaitEvent(es, cx->fork, 0));
            r = launch_class_f64(true, params->pf.n_ins, c, *ka64, poll_ctas(sms), es);
            if (r) return fail(r);
            QP_TRY(cudaEventRecord(cx->join[kNumClasses + (c - kNumPacked)], es));
        }
    }
    prof_mark(cx, 2, st);

    // ---- drainers: what the pollers have not taken when the fp32 classes have finished ----------------------------
    if (refine) {
        k_refine_plan<<<1, 32, 0, st>>>(1, mw64, poll_ctas(sms), avail, (const PairInfo*)(ws + L.info), (const int32_t*)(ws + L.order), hdr);
        ++g_launches;
        QP_TRY(cudaEventRecord(cx->fork2, st));
        ka64->refine_pass = 2;
        for (int c = kNumPacked; c < kSplitEnd; ++c) {
            QP_TRY(cudaStreamWaitEvent(cx->st[c], cx->fork2, 0));
            // every drainer CTA pulls exactly one index past the end of its list (pollers pull none): the pad bounds the grid
            r = launch_class_f64(true, params->pf.n_ins, c, *ka64, std::min(class_grid(c, true, sms), kListPad), cx->st[c]);
            if (r) return fail(r);
            QP_TRY(cudaEventRecord(cx->join[c], cx->st[c]));
        }
    }

    // ---- CSR placement in pair order; it only needs the fp32 pass, so it runs beside the fp64 kernels ------------
    cudaStream_t ps = refine ? cx->st[kNumStreams - 1] : st;
    if (refine) QP_TRY(cudaStreamWaitEvent(ps, cx->fork2, 0));
    scan_launch<int32_t>((const int32_t*)(ws + L.nnz), P, out->pair_nnz_base, (int64_t*)(ws + L.scan_tmp), ps, &g_launches);
    if (out->nnz_capacity > 0)
        k_copy_pool<<<(int)((P + 3) / 4), 128, 0, ps>>>((const int32_t*)(ws + L.nnz), (const int64_t*)(ws + L.pool_off),
                                                        out->pair_nnz_base, P, (const float2*)(ws + L.pool), out->nnz_capacity,
                                                        out->col_idx, out->val);
    if (refine) {
        QP_TRY(cudaEventRecord(cx->join[kNumStreams - 1], ps));
        QP_TRY(cudaStreamWaitEvent(st, cx->join[kNumStreams - 1], 0));
        for (int c = kNumPacked; c < kSplitEnd; ++c) {
            QP_TRY(cudaStreamWaitEvent(st, cx->join[c], 0));                                               // drainers
            if (pollers) QP_TRY(cudaStreamWaitEvent(st, cx->join[kNumClasses + (c - kNumPacked)], 0));     // pollers
        }
    }
    prof_mark(cx, 3, st);
    k_finish<<<1, 32, 0, st>>>(hdr, out->status);
    g_launches += 2;
    prof_mark(cx, 4, st);
    QP_TRY(cudaGetLastError());
#undef QP_TRY

    if (params->flags & QP_FLAG_SYNC_STATUS) {
        int32_t hs[4] = {0, 0, 0, 0};
        QP_CUDA(cudaMemcpyAsync(hs, out->status, sizeof hs, cudaMemcpyDeviceToHost, st));
        QP_CUDA(cudaStreamSynchronize(st));
        return hs[0];
    }
    return QP_OK;
}

extern "C" int qp_posteriors(const uint8_t* d_seqs, const int64_t* d_offsets, int32_t k, const int32_t* d_pairs,
                             int64_t P, const qp_params* params, void* d_workspace, size_t workspace_bytes,
                             const qp_output* out, void* cuda_stream) {
    g_launches = 0;
    if (!out || k < 0 || P < 0 || P > 0x7fffffff) return QP_ERR_INVALID_ARG;
    int r = check_params(params);
    if (r) return r;
    if (!out->pair_row_base || !out->pair_nnz_base || !out->status) return QP_ERR_INVALID_ARG;
    if (P > 0 && (!d_seqs || !d_offsets || !d_pairs || !d_workspace || !out->row_ptr || !out->dist)) return QP_ERR_INVALID_ARG;
    if (out->nnz_capacity < 0 || (out->nnz_capacity > 0 && (!out->col_idx || !out->val))) return QP_ERR_INVALID_ARG;
    if (P > 0 && ((uintptr_t)d_workspace & 255) != 0) return QP_ERR_INVALID_ARG;
    Ctx* cx = ctx_get();
    if (!cx) return QP_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (P == 0) {   // nothing to do: empty prefixes, status ok; the workspace is not touched
        QP_CUDA(cudaMemsetAsync(out->pair_row_base, 0, 8, st));
        QP_CUDA(cudaMemsetAsync(out->pair_nnz_base, 0, 8, st));
        QP_CUDA(cudaMemsetAsync(out->status, 0, 16, st));
        if (params->flags & QP_FLAG_SYNC_STATUS) QP_CUDA(cudaStreamSynchronize(st));
        return QP_OK;
    }
    return run_posteriors(cx, d_seqs, d_offsets, k, d_pairs, P, params, d_workspace, workspace_bytes, out, st);
}

extern "C" int qp_posteriors_budgeted(const uint8_t* d_seqs, const int64_t* d_offsets, int32_t k, const int32_t* d_pairs,
                                      int64_t P, const qp_params* params, void* d_workspace, size_t workspace_bytes,
                                      const qp_output* out, void* cuda_stream, int max_passes, double* tau_used,
                                      int* passes) {
    if (!params || !out || max_passes < 1) return QP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    qp_params prm = *params;
    prm.flags |= QP_FLAG_SYNC_STATUS;
    // pass 1: the stage at the requested threshold, with every kept value counted into threshold bins on the way
    g_want_hist = true;
    g_tau_hist_valid = false;
    int r = qp_posteriors(d_seqs, d_offsets, k, d_pairs, P, &prm, d_workspace, workspace_bytes, out, st);
    g_want_hist = false;
    int launches = g_launches, done = 1;
    if ((r == QP_OK || r == QP_ERR_NNZ_CAPACITY) && P > 0) {
        Ctx* cx = ctx_get();
        const Layout L = make_layout(P, out->nnz_capacity, out->dense_P != nullptr, total_max_slots(cx ? cx->sms : kSmAssumed));
        if (cudaMemcpyAsync(g_tau_hist, (char*)d_workspace + L.tau_hist, sizeof g_tau_hist, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            return QP_ERR_CUDA;
        g_tau0 = (float)prm.threshold;
        g_tau_hist_valid = true;
    }
    if (r == QP_ERR_NNZ_CAPACITY && max_passes >= 2 && g_tau_hist_valid) {
        // the smallest bin edge whose tail of the histogram fits the capacity: exact, the second pass recomputes the
        // very same values
        int32_t bits0;
        memcpy(&bits0, &g_tau0, 4);
        unsigned long long tail = 0;
        int b = kTauBins;              // first bin NOT taken when walking down from the top
        while (b > 0 && tail + g_tau_hist[b - 1] <= (unsigned long long)out->nnz_capacity) tail += g_tau_hist[--b];
        if (b < kTauBins && b > 0) {   // b == 0 cannot happen (the whole histogram did not fit); b == kTauBins: nothing fits
            const int32_t bits = bits0 + (b << kTauShift);
            float tb;
            memcpy(&tb, &bits, 4);
            prm.threshold = (double)tb;
            r = qp_posteriors(d_seqs, d_offsets, k, d_pairs, P, &prm, d_workspace, workspace_bytes, out, st);
            launches += g_launches;
            done = 2;
        }
    }
    g_launches = launches;
    if (tau_used) *tau_used = prm.threshold;
    if (passes) *passes = done;
    return r;
}

extern "C" int qp_last_tau_curve(double* tau, int64_t* count, int max_bins) {
    if (!g_tau_hist_valid || !tau || !count || max_bins < 1) return QP_ERR_INVALID_ARG;
    int32_t bits0;
    memcpy(&bits0, &g_tau0, 4);
    unsigned long long tail = 0;
    const int nb = max_bins < kTauBins ? max_bins : kTauBins;
    for (int b = kTauBins - 1; b >= 0; --b) {
        tail += g_tau_hist[b];
        if (b < nb) {
            const int32_t bits = bits0 + (b << kTauShift);
            float tb;
            memcpy(&tb, &bits, 4);
            tau[b] = (double)tb;
            count[b] = (int64_t)tail;
        }
    }
    return nb;
}
