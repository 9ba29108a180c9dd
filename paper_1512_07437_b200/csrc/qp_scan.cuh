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

}  // namespace qp
