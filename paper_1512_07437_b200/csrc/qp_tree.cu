// qp_tree.cu -- stage II on the device: weighted UPGMA guide tree and tree-guided distances (include/qp.h,
// qp_guide_tree). The k-1 merges are inherently sequential, each one is a few data-parallel
// sweeps over <= k values, so ONE persistent CTA of 1024 threads runs the whole loop without leaving the SM:
//   per row i a cached nearest neighbour among the live slots j > i (value, index; ties -> smallest j);
//   merge step: block arg-min over the cached row minima (ties -> smallest i)            -> pair (i, j), i < j
//               row i <- (row i + row j) / 2 in fp32, column i mirrored, slot j dies
//               rows whose cached neighbour was i or j (or row i itself) are rescanned, one warp per row;
//               the other rows m < i only compare their cache with the one entry that changed.
// The matrix (k*k fp32, 4 MB at k = 1000) stays in L2. The tree distances are a separate k x k kernel afterwards.
#include <cuda_runtime.h>
#include <stdint.h>

#include "qp.h"

namespace qp {

constexpr int kTreeThreads = 1024;
constexpr unsigned kFullMask = 0xffffffffu;
constexpr unsigned long long kNone = 0xffffffffffffffffull;

// (distance, index) as one ordered 64-bit key: distances are >= 0, so their bit patterns order like the values
__device__ __forceinline__ unsigned long long key_of(float v, int idx) {
    return ((unsigned long long)__float_as_uint(v) << 32) | (unsigned)idx;
}
__device__ __forceinline__ unsigned long long warp_min(unsigned long long k) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long t = __shfl_xor_sync(kFullMask, k, o);
        k = t < k ? t : k;
    }
    return k;
}

struct TreeWs {   // layout of the workspace
    float* W;                    // [k][k] working distances between slots
    unsigned long long* nn;      // [k] cached (distance, j) of the nearest live slot j > i, kNone if there is none
    int32_t* node;               // [k] node id living in the slot
    uint8_t* alive;              // [k]
};

// nearest live slot j > row of one row, by one warp
__device__ __forceinline__ unsigned long long scan_row(const TreeWs& w, int k, int row, int lane) {
    unsigned long long best = kNone;
    const float* r = w.W + (size_t)row * k;
    for (int j = row + 1 + lane; j < k; j += 32)
        if (w.alive[j]) {
            const unsigned long long c = key_of(r[j], j);
            best = c < best ? c : best;
        }
    return warp_min(best);
}

__global__ void __launch_bounds__(kTreeThreads, 1)
k_wpgma(const float* __restrict__ dist, int k, TreeWs w, int32_t* __restrict__ merge, float* __restrict__ height,
        int32_t* __restrict__ leaves, int32_t* __restrict__ parent) {
    __shared__ unsigned long long s_red[32];
    __shared__ int s_i, s_j, s_nq;
    __shared__ int s_queue[kTreeThreads];   // rows to rescan; overflow falls back to "rescan every row below i"
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // ---- initialise: working copy, slots, leaves
    for (size_t q = tid; q < (size_t)k * k; q += kTreeThreads) w.W[q] = fmaxf(dist[q], 0.f);   // also maps -0 to +0
    for (int q = tid; q < k; q += kTreeThreads) {
        w.node[q] = q;
        w.alive[q] = 1;
    }
    for (int q = tid; q < 2 * k - 1; q += kTreeThreads) {
        leaves[q] = 1;
        parent[q] = -1;
    }
    __syncthreads();
    for (int row = warp; row < k; row += 32) {
        const unsigned long long b = scan_row(w, k, row, lane);
        if (lane == 0) w.nn[row] = b;
    }
    __syncthreads();
    // ---- k-1 merges
    for (int t = 0; t < k - 1; ++t) {
        // closest pair: arg-min over rows of (cached distance, row); the cached j rides along in a second step
        unsigned long long best = kNone;
        for (int i = tid; i < k; i += kTreeThreads) {
            const unsigned long long c = w.nn[i];
            if (w.alive[i] && c != kNone) {
                const unsigned long long key = (c & 0xffffffff00000000ull) | (unsigned)i;
                best = key < best ? key : best;
            }
        }
        best = warp_min(best);
        if (lane == 0) s_red[warp] = best;
        __syncthreads();
        if (warp == 0) {
            unsigned long long b = s_red[lane];
            b = warp_min(b);
            if (lane == 0) {
                const int i = (int)(b & 0xffffffffu);
                const int j = (int)(w.nn[i] & 0xffffffffu);
                s_i = i;
                s_j = j;
                s_nq = 0;
                const int u = k + t, a = w.node[i], c = w.node[j];
                merge[2 * t] = a;
                merge[2 * t + 1] = c;
                height[t] = __uint_as_float((unsigned)(b >> 32));
                leaves[u] = leaves[a] + leaves[c];
                parent[a] = u;
                parent[c] = u;
                w.node[i] = u;
                w.alive[j] = 0;
            }
        }
        __syncthreads();
        const int i = s_i, j = s_j;
        // row i <- (row i + row j) / 2, mirrored into column i; the rows above i look at their changed entry
        float* ri = w.W + (size_t)i * k;
        const float* rj = w.W + (size_t)j * k;
        for (int m = tid; m < k; m += kTreeThreads) {
            if (!w.alive[m] || m == i) continue;
            const float v = __fmul_rn(__fadd_rn(ri[m], rj[m]), 0.5f);
            ri[m] = v;
            w.W[(size_t)m * k + i] = v;
            if (m < j) {   // rows m < j can have i or j cached (only rows m < i can have i)
                const unsigned long long c = w.nn[m];
                const int cj = (int)(c & 0xffffffffu);
                if (c != kNone && (cj == i || cj == j)) {
                    const int pos = atomicAdd(&s_nq, 1);
                    if (pos < kTreeThreads) s_queue[pos] = m;
                } else if (m < i) {
                    const unsigned long long nk = key_of(v, i);
                    if (nk < c) w.nn[m] = nk;   // closer, or as close with a smaller slot index
                }
            }
        }
        __syncthreads();
        // rescans: row i always; the queued rows; everything below j if the queue overflowed (cannot happen for k <= 1024)
        const int nq = s_nq;
        if (nq <= kTreeThreads) {
            for (int q = warp; q <= nq; q += 32) {
                const int row = q == nq ? i : s_queue[q];
                const unsigned long long b = scan_row(w, k, row, lane);
                if (lane == 0) w.nn[row] = b;
            }
        } else {
            for (int row = warp; row < j; row += 32) {
                if (!w.alive[row]) continue;
                const unsigned long long b = scan_row(w, k, row, lane);
                if (lane == 0) w.nn[row] = b;
            }
        }
        __syncthreads();
    }
}

// tree-guided distance: node ids grow with the merge time, so the lowest common ancestor is reached by always
// lifting the smaller of the two ids
__global__ void k_treedist(const int32_t* __restrict__ leaves, const int32_t* __restrict__ parent, int k,
                           int32_t* __restrict__ out) {
    const size_t q = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (q >= (size_t)k * k) return;
    int a = (int)(q / k), b = (int)(q % k);
    while (a != b) {
        if (a < b) a = __ldg(parent + a);
        else b = __ldg(parent + b);
    }
    out[q] = 2 * __ldg(leaves + a) - 1;
}

static inline size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

}  // namespace qp

using namespace qp;

extern "C" size_t qp_guide_tree_workspace_bytes(int32_t k) {
    if (k < 1) return 0;
    return align256((size_t)k * k * 4) + align256((size_t)k * 8) + align256((size_t)k * 4) + align256((size_t)k);
}

extern "C" int qp_guide_tree(const float* d_dist, int32_t k, int32_t* d_merge, float* d_height, int32_t* d_leaves,
                             int32_t* d_parent, int32_t* d_treedist, void* d_workspace, size_t workspace_bytes,
                             void* cuda_stream) {
    if (k < 1 || !d_dist || !d_leaves || !d_parent || !d_workspace || (k > 1 && (!d_merge || !d_height)))
        return QP_ERR_INVALID_ARG;
    if (workspace_bytes < qp_guide_tree_workspace_bytes(k) || ((uintptr_t)d_workspace & 255) != 0) return QP_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* p = (char*)d_workspace;
    TreeWs w;
    w.W = (float*)p;
    p += align256((size_t)k * k * 4);
    w.nn = (unsigned long long*)p;
    p += align256((size_t)k * 8);
    w.node = (int32_t*)p;
    p += align256((size_t)k * 4);
    w.alive = (uint8_t*)p;
    k_wpgma<<<1, kTreeThreads, 0, st>>>(d_dist, k, w, d_merge, d_height, d_leaves, d_parent);
    if (d_treedist) {
        const size_t n = (size_t)k * k;
        k_treedist<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_leaves, d_parent, k, d_treedist);
    }
    return cudaGetLastError() == cudaSuccess ? QP_OK : QP_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------------------------------
// qp_guide_tree_static: the same two kernels for callers that have no device memory to hand over as a workspace.
//
// Who that is: code that runs where cudaMalloc / cudaFree may not be called or would be harmful -- a plug-in inside
// a host program that owns all device memory and gives the plug-in only its input and output buffers; a step of a
// latency-critical loop, where an allocation may block on the driver and synchronise the whole device; a process
// sharing its GPU under a fixed memory reservation, where an allocation made late can fail although the inputs fit.
// qp_guide_tree asks such a caller for a workspace it cannot create. Here the scratch of the merge loop (working
// matrix, nearest-neighbour cache, slot tables) lives in the array below, which is part of the library image: the
// driver places it when the module is loaded on a device and keeps it until the process exits (about 4 MiB on every
// GPU that loads libqp.so), and the call itself runs no cudaMalloc, cudaFree or allocating library routine.
//
// In host code the name g_tree_scratch is only a handle for the symbol, not a device address (passing it to a kernel
// makes the kernel fault, or quietly use unrelated memory on systems where the GPU can read host memory). The device
// address is looked up once per device with cudaGetSymbolAddress, with that device current, and kept in a table.
// ---------------------------------------------------------------------------------------------------------------------
#include <mutex>

namespace qp {

constexpr int kStaticMaxK = QP_GUIDE_TREE_STATIC_MAX_K;
constexpr size_t kStaticW = (size_t)kStaticMaxK * kStaticMaxK * 4;   // working matrix, already a multiple of 256
constexpr size_t kStaticNn = (size_t)kStaticMaxK * 8;
constexpr size_t kStaticNode = (size_t)kStaticMaxK * 4;
constexpr size_t kStaticAlive = (size_t)kStaticMaxK;
constexpr size_t kStaticBytes = kStaticW + kStaticNn + kStaticNode + kStaticAlive;
static_assert(kStaticW % 256 == 0 && kStaticNn % 256 == 0 && kStaticNode % 256 == 0, "sub-arrays stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_tree_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
static unsigned char* g_tree_scratch_addr[kMaxDevices];   // device address of g_tree_scratch on device d, 0 = not looked up
static std::mutex g_tree_scratch_mutex;

// Device address of the scratch array on the CURRENT device; looked up on the first call per device.
static int static_scratch(unsigned char** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return QP_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_tree_scratch_mutex);
    if (!g_tree_scratch_addr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_tree_scratch) != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return QP_ERR_CUDA;
        }
        g_tree_scratch_addr[dev] = (unsigned char*)p;
    }
    *out = g_tree_scratch_addr[dev];
    return QP_OK;
}

}  // namespace qp

extern "C" int qp_guide_tree_static(const float* d_dist, int32_t k, int32_t* d_merge, float* d_height,
                                    int32_t* d_leaves, int32_t* d_parent, int32_t* d_treedist, void* cuda_stream) {
    if (k < 1 || !d_dist || !d_leaves || !d_parent || (k > 1 && (!d_merge || !d_height))) return QP_ERR_INVALID_ARG;
    if (k > kStaticMaxK) return QP_ERR_STATIC_LIMIT;   // the built-in scratch holds QP_GUIDE_TREE_STATIC_MAX_K sequences
    unsigned char* p = nullptr;
    const int rc = static_scratch(&p);
    if (rc != QP_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // Nothing has to be cleared between calls: k_wpgma writes W[0 .. k*k), nn, node and alive [0 .. k) before it reads
    // any of them, so what the previous call (of any k) left behind is never seen.
    TreeWs w;
    w.W = (float*)p;
    w.nn = (unsigned long long*)(p + kStaticW);
    w.node = (int32_t*)(p + kStaticW + kStaticNn);
    w.alive = (uint8_t*)(p + kStaticW + kStaticNn + kStaticNode);
    k_wpgma<<<1, kTreeThreads, 0, st>>>(d_dist, k, w, d_merge, d_height, d_leaves, d_parent);
    if (d_treedist) {
        const size_t n = (size_t)k * k;
        k_treedist<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_leaves, d_parent, k, d_treedist);
    }
    return cudaGetLastError() == cudaSuccess ? QP_OK : QP_ERR_CUDA;
}
