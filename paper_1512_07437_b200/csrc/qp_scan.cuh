// qp_scan.cuh -- small prefix-sum helpers shared by the scheduling kernels (qp_api.cu) and stage III (qp_consistency.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qp {

// block-wide exclusive scan of one value per thread (1024 threads), returns the exclusive prefix; total in *tot
__device__ inline int64_t block_excl_scan(int64_t v, int64_t* sh, int64_t* tot) {
    const int t = threadIdx.x;
    sh[t] = v;
    __syncthreads();
    for (int o = 1; o < (int)blockDim.x; o <<= 1) {
        int64_t a = (t >= o) ? sh[t - o] : 0;
        __syncthreads();
        sh[t] += a;
        __syncthreads();
    }
    int64_t incl = sh[t];
    *tot = sh[blockDim.x - 1];
    __syncthreads();
    return incl - v;
}

// out[0..P] = exclusive prefix of in[0..P-1]; single block
template <typename T> __global__ void k_scan(const T* __restrict__ in, int64_t P, int64_t* __restrict__ out) {
    __shared__ int64_t sh[1024];
    const int t = threadIdx.x;
    const int64_t per = (P + blockDim.x - 1) / blockDim.x;
    const int64_t lo = min(P, t * per), hi = min(P, (t + 1) * per);
    int64_t loc = 0;
    for (int64_t q = lo; q < hi; ++q) loc += (int64_t)in[q];
    int64_t tot;
    int64_t ex = block_excl_scan(loc, sh, &tot);
    for (int64_t q = lo; q < hi; ++q) {
        out[q] = ex;
        ex += (int64_t)in[q];
    }
    if (t == 0) out[P] = tot;
}

// The same prefix over many blocks, for long inputs (one block walks 5e5 values in 0.64 ms, mostly waiting on its own
// strided loads): every block of kScanChunk values is summed (k_scan_sums), the block sums are scanned by one block
// (k_scan), every block then scans its own values onto its offset (k_scan_apply). `sums` holds nblk + 1 int64.
constexpr int kScanChunk = 4096;   // values per block: 1024 threads x 4
template <typename T> __global__ void k_scan_sums(const T* __restrict__ in, int64_t P, int64_t* __restrict__ sums) {
    __shared__ int64_t sh[32];
    const int64_t base = (int64_t)blockIdx.x * kScanChunk;
    int64_t v = 0;
    for (int q = threadIdx.x; q < kScanChunk; q += blockDim.x)
        if (base + q < P) v += (int64_t)in[base + q];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) sums[blockIdx.x] = v;
    }
}
template <typename T>
__global__ void k_scan_apply(const T* __restrict__ in, int64_t P, const int64_t* __restrict__ offs /*exclusive prefix of the block sums*/,
                             int64_t nblk, int64_t* __restrict__ out) {
    __shared__ int64_t sh[1024];
    const int64_t base = (int64_t)blockIdx.x * kScanChunk;
    const int t = threadIdx.x;
    // thread t owns 4 consecutive values: loads of a warp cover 512 contiguous bytes (int32) per round of 4
    int64_t v[4], loc = 0;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int64_t q = base + 4 * t + u;
        v[u] = q < P ? (int64_t)in[q] : 0;
        loc += v[u];
    }
    int64_t tot;
    int64_t ex = block_excl_scan(loc, sh, &tot) + offs[blockIdx.x];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int64_t q = base + 4 * t + u;
        if (q < P) out[q] = ex;
        ex += v[u];
    }
    if (blockIdx.x == nblk - 1 && t == 0) out[P] = offs[nblk];
}
// host helper: out[0..P] = exclusive prefix of in[0..P-1]; `sums` = scratch of (P / kScanChunk + 2) * 2 int64
template <typename T> inline void scan_launch(const T* in, int64_t P, int64_t* out, int64_t* sums, cudaStream_t st, int* launches) {
    if (P <= 8 * kScanChunk) {   // short: one block is as fast and one launch instead of three
        k_scan<T><<<1, 1024, 0, st>>>(in, P, out);
        if (launches) *launches += 1;
        return;
    }
    const int64_t nblk = (P + kScanChunk - 1) / kScanChunk;
    int64_t* offs = sums + nblk + 1;
    k_scan_sums<T><<<(int)nblk, 256, 0, st>>>(in, P, sums);
    k_scan<int64_t><<<1, 1024, 0, st>>>(sums, nblk, offs);
    k_scan_apply<T><<<(int)nblk, 1024, 0, st>>>(in, P, offs, nblk, out);
    if (launches) *launches += 3;
}

}  // namespace qp
